"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

EVERY output site is compared with the oracle: a full even-parity pass of the oracle costs 66 ms at 32^3x64 and
under half a second at 48^3x96 on the box's host cores (bench.py's cpu_baseline does 180 of them), so nothing is
sampled.  Solves are judged by their true residual with the oracle's operator (one full-lattice oracle apply).
Inputs: the seeded recipes of DESIGN.md §4.
"""
import numpy as np
import pytest

from oracle import bqo
from paper_2111_04457_b200 import inputs
from tests.conftest import relmax

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2111_04457_b200 import bq as _bq
    _bq.lib()
    return _bq


def even_sites_of(L):
    return np.nonzero(inputs.site_parity(L).ravel() == 0)[0]


def oracle_even_hop(U, psi, kappa, L):
    """-kappa H_eo psi_o at ALL even sites: (D [0; psi_odd])(x), x even -> [Vh, 4, 3] (oracle, site by site)."""
    masked = np.where((inputs.site_parity(L) == 1)[..., None, None], psi, 0)
    return bqo.dirac_apply_sites(U, masked, kappa, even_sites_of(L))


def test_config2_16to4_fp32_apply_1000x(bq):
    """BASELINE.json config 2: 16^4, fp32, 18-real, kappa = 0.125; 1000 back-to-back applies (reading S12)."""
    import torch
    L = (16, 16, 16, 16)
    seed = inputs.BASE_SEED + 2
    U, psi = inputs.gauge(L, seed, 0.3), inputs.spinor(L, seed)
    ref = bqo.hop_restricted(U, psi, 0.125, 0)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        src = lat.import_field(psi, bq.BQ_FP32, bq.BQ_ODD)
        out = lat.field(bq.BQ_FP32, bq.BQ_EVEN)
        bq.bq_wilson_apply(lat.h, out, src, 0.125, bq.BQ_EVEN, bq.BQ_FP32, bq.BQ_RECON18)
        first = out.clone()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for _ in range(999):
            bq.bq_wilson_apply(lat.h, out, src, 0.125, bq.BQ_EVEN, bq.BQ_FP32, bq.BQ_RECON18)
        ev1.record()
        torch.cuda.synchronize()
        assert torch.equal(first, out)                       # 1st and 1000th bitwise identical
        assert relmax(lat.export_field(out, bq.BQ_FP32, bq.BQ_EVEN), ref) < 1e-5
        us = ev0.elapsed_time(ev1) / 999 * 1e3
        print(f"config 2: {us:.2f} us per apply (L2-resident working set: not an HBM measurement), "
              f"{1320 * 32768 / us / 1e3:.0f} GFlop/s")


def test_config3_32x32x32x64_hop_every_site(bq):
    """BASELINE.json config 3: 32^3x64 even-odd hop, eps = 0.5 — the bench workload — fp32 with 18- and 12-real links
    (1e-5), fp64 (1e-12) and half storage (5e-3): all 1,048,576 output sites against the oracle."""
    L = (32, 32, 32, 64)
    seed = inputs.BASE_SEED + 3
    U, psi = inputs.gauge(L, seed, 0.5), inputs.spinor(L, seed)
    ev = even_sites_of(L)
    ref = oracle_even_hop(U, psi, 0.125, L)
    odd = inputs.site_parity(L).ravel() == 1
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        for prec, recon, tol in ((bq.BQ_FP32, 0, 1e-5), (bq.BQ_FP32, 1, 1e-5), (bq.BQ_FP64, 0, 1e-12), (bq.BQ_FP64, 1, 1e-12),
                                 (bq.BQ_HALF, 0, 5e-3), (bq.BQ_HALF, 1, 5e-3)):
            src = lat.import_field(psi, prec, bq.BQ_ODD)
            out = lat.field(prec, bq.BQ_EVEN)
            bq.bq_wilson_apply(lat.h, out, src, 0.125, bq.BQ_EVEN, prec, recon)
            got = lat.export_field(out, prec, bq.BQ_EVEN).reshape(-1, 4, 3)
            err = relmax(got[ev], ref)
            print(f"config 3 prec={prec} recon={recon}: max rel err over {len(ev)} sites {err:.2e}")
            assert err < tol, (prec, recon)
            assert np.all(got[odd] == 0)                     # the export leaves the other parity alone
            del src, out


def test_config3_multirhs_x12_every_site(bq):
    """32^3 x 64 fp32, half and fp64 storage, 12 right-hand sides in one launch (the link-stationary kernels, as bench.py --kernels and
    bench.py time them: hop_ls.cuh for fp32 / half, the direction-split hop_lsp.cuh for fp64): every output site of every
    right-hand side against the oracle, and every right-hand side bit for bit against the single-rhs kernel."""
    import torch
    L, kappa, nrhs = (32, 32, 32, 64), 0.125, 12
    seed = inputs.BASE_SEED + 3
    U = inputs.gauge(L, seed, 0.5)
    psis = [inputs.spinor(L, seed + 1000 * k) for k in range(nrhs)]
    ev = even_sites_of(L)
    refs = [oracle_even_hop(U, p, kappa, L) for p in psis]
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        for prec, tol in ((bq.BQ_FP32, 1e-5), (bq.BQ_HALF, 5e-3), (bq.BQ_FP64, 1e-12)):
            fb = bq.bq_field_bytes(lat.h, prec, bq.BQ_EVEN)
            src = torch.cat([lat.import_field(p, prec, bq.BQ_ODD) for p in psis])
            out = torch.zeros(nrhs * fb, dtype=torch.uint8, device="cuda")
            one = lat.field(prec, bq.BQ_EVEN)
            for recon in (bq.BQ_RECON18, bq.BQ_RECON12):
                c0 = bq.bq_get_counters(lat.h)
                bq.bq_wilson_apply_multi(lat.h, out, src, nrhs, kappa, bq.BQ_EVEN, prec, recon)
                c1 = bq.bq_get_counters(lat.h)
                assert c1["ls"] == c0["ls"] + 1 and c1["lsp"] == c0["lsp"] + (1 if prec == bq.BQ_FP64 else 0)
                for k in range(nrhs):
                    bq.bq_wilson_apply(lat.h, one, src[k * fb:(k + 1) * fb], kappa, bq.BQ_EVEN, prec, recon)
                    assert torch.equal(one, out[k * fb:(k + 1) * fb]), (prec, recon, k)
                    if recon == bq.BQ_RECON18 or k in (0, 11):
                        got = lat.export_field(out[k * fb:(k + 1) * fb], prec, bq.BQ_EVEN).reshape(-1, 4, 3)[ev]
                        assert relmax(got, refs[k]) < tol, (prec, recon, k)
            del src, out


@pytest.fixture(scope="module")
def config4():
    """Gauge field, source and the oracle's dense clover term (and its inverse) of BASELINE config 4."""
    L = (32, 32, 32, 64)
    seed = inputs.BASE_SEED + 4
    csw, kappa = 1.0, 0.1215
    U, b = inputs.gauge(L, seed, 0.5), inputs.spinor(L, seed)
    A = bqo.clover_build(U, csw, kappa)
    return L, csw, kappa, U, b, A


def test_config4_clover_operator_every_site(bq, config4):
    """32^3x64 Wilson-clover D (bq_dirac_apply, csw = 1) and its even-odd Schur complement (bq_schur_apply) on the
    whole lattice against the oracle's dense-clover operator: fp32 <= 1e-5 / 2e-5 (two hops), fp64 <= 1e-12 / 2e-12."""
    import torch
    L, csw, kappa, U, psi, A = config4
    ref = bqo.dirac_apply(U, psi, kappa, A=A)
    par = (inputs.site_parity(L) == 0)[..., None, None]
    Ainv = bqo.site_matrix_invert(A)
    ref_s = bqo.schur_apply(U, np.where(par, psi, 0), kappa, A=A, Ainv=Ainv)
    del Ainv
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        for prec, tol in ((bq.BQ_FP32, 1e-5), (bq.BQ_FP64, 1e-12)):
            src = lat.import_field(psi, prec, bq.BQ_FULL)
            out = torch.zeros_like(src)
            bq.bq_dirac_apply(lat.h, out, src, kappa, csw, prec, bq.BQ_RECON18)
            err = relmax(lat.export_field(out, prec, bq.BQ_FULL), ref)
            src_e = lat.import_field(psi, prec, bq.BQ_EVEN)
            out_e, tmp = torch.zeros_like(src_e), torch.zeros_like(src_e)
            bq.bq_schur_apply(lat.h, out_e, src_e, tmp, kappa, csw, prec, bq.BQ_RECON18)
            err_s = relmax(lat.export_field(out_e, prec, bq.BQ_EVEN), ref_s)
            print(f"config 4 prec={prec}: D {err:.2e}, Schur {err_s:.2e} (all {psi.size // 12} sites)")
            assert err < tol and err_s < 2 * tol, prec
            del src, out, src_e, out_e, tmp


def test_config4_clover_solve_32x32x32x64(bq, config4):
    """BASELINE.json config 4: Wilson-clover csw = 1, kappa = 0.1215, fp32 inner / fp64 outer BiCGStab to 1e-10."""
    L, csw, kappa, U, b, A = config4
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        info = bq.bq_solve(lat.h, b, x, kappa, 1e-10, bq.bq_solve_opts(inner_prec=bq.BQ_FP32, csw=csw))
        c = bq.bq_get_counters(lat.h)
    res = np.linalg.norm(b - bqo.dirac_apply(U, x, kappa, A=A)) / np.linalg.norm(b)
    print(f"config 4: {info.inner_iters} inner iters, {info.outer_cycles} outer, {info.seconds * 1e3:.1f} ms, "
          f"oracle residual {res:.2e}, hops {c['hop_fp32']} launched / {c['idle_fp32']} no-ops after convergence")
    assert info.status == 0 and res <= 1e-10
    # hops enqueued after convergence are accounted for: 4 per launched-but-unused iteration
    assert c["idle_fp32"] % 4 == 0 and c["hop_fp32"] - c["idle_fp32"] == 4 * info.inner_iters


def test_config5_half_solve_48x48x48x96(bq):
    """BASELINE.json config 5: 48^3x96 Wilson, kappa = 0.1235, eps = 0.7, half-storage inner, fp64 outer, to 1e-10;
    and the half-storage hop at that size on every one of its 5,308,416 output sites (5e-3)."""
    L = (48, 48, 48, 96)
    seed = inputs.BASE_SEED + 5
    kappa = 0.1235
    U, b = inputs.gauge(L, seed, 0.7), inputs.spinor(L, seed)
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        info = bq.bq_solve(lat.h, b, x, kappa, 1e-10, bq.bq_solve_opts(inner_prec=bq.BQ_HALF))
        ev = even_sites_of(L)
        ref = oracle_even_hop(U, b, kappa, L)
        src = lat.import_field(b, bq.BQ_HALF, bq.BQ_ODD)
        out = lat.field(bq.BQ_HALF, bq.BQ_EVEN)
        bq.bq_wilson_apply(lat.h, out, src, kappa, bq.BQ_EVEN, bq.BQ_HALF, bq.BQ_RECON18)
        got = lat.export_field(out, bq.BQ_HALF, bq.BQ_EVEN).reshape(-1, 4, 3)
        err = relmax(got[ev], ref)
        print(f"config 5 half hop: max rel err over {len(ev)} sites {err:.2e}")
        assert err < 5e-3
    res = np.linalg.norm(b - bqo.dirac_apply(U, x, kappa)) / np.linalg.norm(b)
    print(f"config 5: {info.inner_iters} inner iters, {info.outer_cycles} outer, {info.seconds * 1e3:.1f} ms, "
          f"oracle residual {res:.2e}")
    assert info.status == 0 and res <= 1e-10
