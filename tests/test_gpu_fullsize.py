"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

The oracle cannot afford many full passes at these sizes, so the hop is checked on sampled output sites the
oracle computes one by one (oracle dirac_apply_sites), and solves by their true residual with the oracle's
operator (one full-lattice oracle apply).  Inputs: the seeded recipes of DESIGN.md §4.
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


def sample_sites(L, parity, n, seed):
    par = inputs.site_parity(L).ravel()
    sites = np.nonzero(par == parity)[0]
    rng = np.random.default_rng(seed)
    pick = rng.choice(sites, size=n, replace=False)
    # always include the corners of the index range and of the lattice (wrap in every direction)
    Lx, Ly, Lz, Lt = L
    corners = [0 if parity == 0 else 1, sites[-1], sites[len(sites) // 2]]
    return np.unique(np.concatenate([pick, np.array(corners)]))


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


@pytest.mark.parametrize("recon", [0, 1])
def test_config3_32x32x32x64_fp32_hop_sampled(bq, recon):
    """BASELINE.json config 3: 32^3x64 fp32 even-odd hop, 18- and 12-real links, eps = 0.5 — the bench workload."""
    L = (32, 32, 32, 64)
    seed = inputs.BASE_SEED + 3
    U, psi = inputs.gauge(L, seed, 0.5), inputs.spinor(L, seed)
    masked = np.where((inputs.site_parity(L) == 1)[..., None, None], psi, 0)
    sites = sample_sites(L, 0, 4096, 3)
    ref = bqo.dirac_apply_sites(U, masked, 0.125, sites)      # even sites, odd-only input: exactly -kappa H_eo psi_o
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        src = lat.import_field(psi, bq.BQ_FP32, bq.BQ_ODD)
        out = lat.field(bq.BQ_FP32, bq.BQ_EVEN)
        bq.bq_wilson_apply(lat.h, out, src, 0.125, bq.BQ_EVEN, bq.BQ_FP32, recon)
        got = lat.export_field(out, bq.BQ_FP32, bq.BQ_EVEN).reshape(-1, 4, 3)
        assert relmax(got[sites], ref) < 1e-5
        # properties that hold at any size: odd sites untouched (zero), output finite, norm consistent with the sample
        odd = inputs.site_parity(L).ravel() == 1
        assert np.all(got[odd] == 0) and np.all(np.isfinite(got.view(np.float64)))
        # linearity on the whole field: H(2 psi) = 2 H(psi) exactly in binary floating point
        src2 = lat.import_field(2 * psi, bq.BQ_FP32, bq.BQ_ODD)
        out2 = lat.field(bq.BQ_FP32, bq.BQ_EVEN)
        bq.bq_wilson_apply(lat.h, out2, src2, 0.125, bq.BQ_EVEN, bq.BQ_FP32, recon)
        assert np.array_equal(lat.export_field(out2, bq.BQ_FP32, bq.BQ_EVEN).reshape(-1, 4, 3), 2 * got)


def test_config4_clover_solve_32x32x32x64(bq):
    """BASELINE.json config 4: Wilson-clover csw = 1, kappa = 0.1215, fp32 inner / fp64 outer BiCGStab to 1e-10."""
    L = (32, 32, 32, 64)
    seed = inputs.BASE_SEED + 4
    csw, kappa = 1.0, 0.1215
    U, b = inputs.gauge(L, seed, 0.5), inputs.spinor(L, seed)
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        info = bq.bq_solve(lat.h, b, x, kappa, 1e-10, bq.bq_solve_opts(inner_prec=bq.BQ_FP32, csw=csw))
    A = bqo.clover_build(U, csw, kappa)
    res = np.linalg.norm(b - bqo.dirac_apply(U, x, kappa, A=A)) / np.linalg.norm(b)
    print(f"config 4: {info.inner_iters} inner iters, {info.outer_cycles} outer, {info.seconds * 1e3:.1f} ms, "
          f"oracle residual {res:.2e}")
    assert info.status == 0 and res <= 1e-10


def test_config5_half_solve_48x48x48x96(bq):
    """BASELINE.json config 5: 48^3x96 Wilson, kappa = 0.1235, eps = 0.7, half-storage inner, fp64 outer, to 1e-10."""
    L = (48, 48, 48, 96)
    seed = inputs.BASE_SEED + 5
    kappa = 0.1235
    U, b = inputs.gauge(L, seed, 0.7), inputs.spinor(L, seed)
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        info = bq.bq_solve(lat.h, b, x, kappa, 1e-10, bq.bq_solve_opts(inner_prec=bq.BQ_HALF))
        # half hop at full size on sampled sites (5e-3)
        masked = np.where((inputs.site_parity(L) == 1)[..., None, None], b, 0)
        sites = sample_sites(L, 0, 2048, 5)
        ref = bqo.dirac_apply_sites(U, masked, kappa, sites)
        src = lat.import_field(b, bq.BQ_HALF, bq.BQ_ODD)
        out = lat.field(bq.BQ_HALF, bq.BQ_EVEN)
        bq.bq_wilson_apply(lat.h, out, src, kappa, bq.BQ_EVEN, bq.BQ_HALF, bq.BQ_RECON18)
        got = lat.export_field(out, bq.BQ_HALF, bq.BQ_EVEN).reshape(-1, 4, 3)
        assert relmax(got[sites], ref) < 5e-3
    res = np.linalg.norm(b - bqo.dirac_apply(U, x, kappa)) / np.linalg.norm(b)
    print(f"config 5: {info.inner_iters} inner iters, {info.outer_cycles} outer, {info.seconds * 1e3:.1f} ms, "
          f"oracle residual {res:.2e}")
    assert info.status == 0 and res <= 1e-10


def test_config3_multirhs_x12_sampled(bq):
    """32^3 x 64 fp32 (BASELINE config 3 shape), 12 right-hand sides in one launch (the patch-mapped multi-rhs kernel, as
    kbench times it): sampled output sites of every right-hand side against the oracle, and the first right-hand side
    bit for bit against the single-rhs kernel."""
    import torch
    L, kappa, nrhs = (32, 32, 32, 64), 0.125, 12
    seed = inputs.BASE_SEED + 3
    U = inputs.gauge(L, seed, 0.5)
    psis = [inputs.spinor(L, seed + 1000 * k) for k in range(nrhs)]
    par = inputs.site_parity(L)
    sites = sample_sites(L, 0, 256, 17)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        fb = bq.bq_field_bytes(lat.h, bq.BQ_FP32, bq.BQ_EVEN)
        src = torch.cat([lat.import_field(p, bq.BQ_FP32, bq.BQ_ODD) for p in psis])
        out = torch.zeros(nrhs * fb, dtype=torch.uint8, device="cuda")
        for recon in (bq.BQ_RECON18, bq.BQ_RECON12):
            bq.bq_wilson_apply_multi(lat.h, out, src, nrhs, kappa, bq.BQ_EVEN, bq.BQ_FP32, recon)
            one = lat.field(bq.BQ_FP32, bq.BQ_EVEN)
            bq.bq_wilson_apply(lat.h, one, src[:fb], kappa, bq.BQ_EVEN, bq.BQ_FP32, recon)
            assert torch.equal(one, out[:fb])
            for k in range(nrhs):
                got = lat.export_field(out[k * fb:(k + 1) * fb], bq.BQ_FP32, bq.BQ_EVEN).reshape(-1, 4, 3)[sites]
                masked = np.where((par == 1)[..., None, None], psis[k], 0)
                ref = bqo.dirac_apply_sites(U, masked, kappa, sites)
                assert relmax(got, ref) < 1e-5, (recon, k)
