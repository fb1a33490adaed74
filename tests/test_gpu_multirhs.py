"""GPU parity of the multi-right-hand-side kernels (the 12 spin-colour
sources of a propagator share one gauge field): every right-hand side against the CPU oracle element by element, and
against the single-rhs kernel bit for bit (same per-site arithmetic, another thread mapping)."""
import numpy as np
import pytest

from oracle import bqo
from paper_2111_04457_b200 import inputs
from tests.conftest import relmax

pytestmark = pytest.mark.gpu

TOL = {0: 1e-12, 1: 1e-5, 2: 5e-3}
GENERAL_BC = np.exp(1j * np.array([0.4, -1.3, 2.0, 0.9]))


@pytest.fixture(scope="module")
def bq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2111_04457_b200 import bq as _bq
    _bq.lib()
    return _bq


def rhs_set(L, n, seed):
    return [inputs.spinor(L, seed + 100 * k) for k in range(n)]


def import_multi(bq, lat, psis, prec, parity):
    import torch
    return torch.cat([lat.import_field(p, prec, parity) for p in psis])


def export_multi(bq, lat, buf, n, prec, parity):
    fb = bq.bq_field_bytes(lat.h, prec, parity)
    return [lat.export_field(buf[k * fb:(k + 1) * fb], prec, parity) for k in range(n)]


# nrhs: 1 (degenerate), 3 and 5 (CTA padded to whole warps, warps cut across tiles), 4, 12 (the propagator), 16 (the most
# one launch holds), 19 (two chunks of 10 + 9).  Lattices: several CTAs with a ragged last CTA; an L = 2 direction.
@pytest.mark.parametrize("L", [(8, 4, 6, 4), (6, 6, 4, 10), (4, 2, 6, 2)])
@pytest.mark.parametrize("prec", [0, 1, 2])
@pytest.mark.parametrize("nrhs", [1, 3, 4, 5, 12, 16, 19])
def test_hop_multi_parity(bq, L, prec, nrhs):
    import torch
    kappa = 0.125
    U = inputs.gauge(L, 61, 0.5)
    psis = rhs_set(L, nrhs, 62)
    recon = nrhs % 2          # alternate 18- and 12-real links over the cases
    for bc in (None, GENERAL_BC):
        with bq.Lattice(L, bc) as lat:
            bq.bq_gauge_load(lat.h, U)
            for p in (0, 1):
                src = import_multi(bq, lat, psis, prec, 1 - p)
                fb = bq.bq_field_bytes(lat.h, prec, p)
                out = torch.zeros(nrhs * fb, dtype=torch.uint8, device="cuda")
                bq.bq_wilson_apply_multi(lat.h, out, src, nrhs, kappa, p, prec, recon)
                got = export_multi(bq, lat, out, nrhs, prec, p)
                one = lat.field(prec, p)
                for k in range(nrhs):
                    ref = bqo.hop_restricted(U, psis[k], kappa, p, bc=bc)
                    assert relmax(got[k], ref) < TOL[prec], (L, prec, nrhs, k, p)
                    bq.bq_wilson_apply(lat.h, one, src[k * fb:(k + 1) * fb], kappa, p, prec, recon)
                    assert torch.equal(one, out[k * fb:(k + 1) * fb]), (L, prec, nrhs, k, p)


@pytest.mark.parametrize("prec", [0, 1, 2])
def test_full_apply_multi(bq, prec):
    import torch
    L, kappa, nrhs = (8, 4, 6, 4), 0.12, 6
    U = inputs.gauge(L, 63, 0.3)
    psis = rhs_set(L, nrhs, 64)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        src = import_multi(bq, lat, psis, prec, bq.BQ_FULL)
        out = torch.zeros_like(src)
        bq.bq_wilson_apply_multi(lat.h, out, src, nrhs, kappa, bq.BQ_FULL, prec, bq.BQ_RECON18)
        for k, got in enumerate(export_multi(bq, lat, out, nrhs, prec, bq.BQ_FULL)):
            assert relmax(got, bqo.dirac_apply(U, psis[k], kappa)) < TOL[prec], k


@pytest.mark.parametrize("prec", [0, 1, 2])
@pytest.mark.parametrize("csw", [0.0, 1.0])
def test_schur_multi_parity(bq, prec, csw):
    import torch
    L, kappa, nrhs = (8, 4, 6, 4), 0.1215, 12
    U = inputs.gauge(L, 65, 0.5)
    psis = rhs_set(L, nrhs, 66)
    A = bqo.clover_build(U, csw, kappa) if csw else None
    Ainv = bqo.site_matrix_invert(A) if csw else None
    par = (inputs.site_parity(L) == 0)[..., None, None]
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        src = import_multi(bq, lat, psis, prec, bq.BQ_EVEN)
        out, tmp = torch.zeros_like(src), torch.zeros_like(src)
        bq.bq_schur_apply_multi(lat.h, out, src, tmp, nrhs, kappa, csw, prec)
        for k, got in enumerate(export_multi(bq, lat, out, nrhs, prec, bq.BQ_EVEN)):
            ref = bqo.schur_apply(U, np.where(par, psis[k], 0), kappa, A=A, Ainv=Ainv)
            assert relmax(got, ref) < 2 * TOL[prec], (prec, csw, k)     # two hops


# ---------------------------------------------------------------------------------------------------
# batched solve (bq_solve_multi): every right-hand side judged with the ORACLE's operator
# ---------------------------------------------------------------------------------------------------
def oracle_residual(U, x, b, kappa, A=None):
    return np.linalg.norm(b - bqo.dirac_apply(U, x, kappa, A=A)) / np.linalg.norm(b)


@pytest.mark.parametrize("inner,csw,nrhs", [(0, 0.0, 3), (1, 0.0, 12), (1, 1.0, 12), (2, 0.0, 5), (1, 1.0, 1), (2, 1.0, 4)])
def test_solve_multi(bq, inner, csw, nrhs):
    """The 12 spin-colour point sources of a propagator for nrhs = 12, Gaussian sources otherwise;
    one right-hand side is zero and one is tiny to exercise the per-rhs stopping logic."""
    L = (8, 4, 8, 8)
    kappa = 0.1215
    U = inputs.gauge(L, 67, 0.5)
    A = bqo.clover_build(U, csw, kappa) if csw else None
    if nrhs == 12:
        b = np.zeros((12,) + (L[3], L[2], L[1], L[0], 4, 3), dtype=np.complex128)
        for s in range(4):
            for c in range(3):
                b[3 * s + c, 0, 0, 0, 0, s, c] = 1.0
    else:
        b = np.stack(rhs_set(L, nrhs, 68))
        if nrhs >= 3:
            b[1] = 0
            b[2] *= 1e-6
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        opts = bq.bq_solve_opts(inner_prec=inner, csw=csw)
        infos = bq.bq_solve_multi(lat.h, b, x, nrhs, kappa, 1e-10, opts)
        # the batched solve and nrhs separate solves agree (same mathematics per right-hand side)
        x1 = np.zeros_like(b[0])
        info1 = bq.bq_solve(lat.h, b[0], x1, kappa, 1e-10, opts)
    assert len(infos) == nrhs
    for k in range(nrhs):
        assert infos[k].status == 0
        if not b[k].any():
            assert not x[k].any() and infos[k].inner_iters == 0
            continue
        res = oracle_residual(U, x[k], b[k], kappa, A=A)
        assert res <= 1e-10 and abs(res - infos[k].true_rel_residual) < 1e-11, (k, res)
    assert np.linalg.norm(x[0] - x1) / np.linalg.norm(x1) < 1e-9
    assert infos[0].inner_iters == info1.inner_iters
    print(f"inner={inner} csw={csw} nrhs={nrhs}: iters {[i.inner_iters for i in infos]} outer {[i.outer_cycles for i in infos]}")


def test_solve_multi_device_buffers_and_errors(bq):
    import torch
    L, kappa, nrhs = (4, 4, 4, 4), 0.12, 2
    U = inputs.gauge(L, 69, 0.3)
    b = np.stack(rhs_set(L, nrhs, 70))
    bd = torch.from_numpy(b).cuda()
    xd = torch.zeros_like(bd)
    with bq.Lattice(L) as lat:
        with pytest.raises(bq.BqError):
            bq.bq_solve_multi(lat.h, bd, xd, nrhs, kappa, 1e-10)        # no gauge field yet
        bq.bq_gauge_load(lat.h, U)
        with pytest.raises(bq.BqError):
            bq.bq_solve_multi(lat.h, bd, xd, 0, kappa, 1e-10)
        infos = bq.bq_solve_multi(lat.h, bd, xd, nrhs, kappa, 1e-10)
        x = xd.cpu().numpy()
        for k in range(nrhs):
            assert oracle_residual(U, x[k], b[k], kappa) <= 1e-10
        opts = bq.bq_solve_opts(inner_prec=bq.BQ_FP32, max_inner=2, max_outer=2, check_every=1)
        xd.zero_()
        infos = bq.bq_solve_multi(lat.h, bd, xd, nrhs, kappa, 1e-12, opts, raise_on_fail=False)
        assert all(i.status == bq.BQ_ENOTCONVERGED for i in infos)


# ---------------------------------------------------------------------------------------------------
# patch mapping of the multi-rhs hop (4 rhs x 2 x 2 tiles per CTA; taken when the x-rows hold whole tiles, Lx % 16 == 0)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [(16, 4, 4, 4), (32, 6, 8, 2), (16, 2, 6, 4)])
@pytest.mark.parametrize("prec", [0, 1, 2])
@pytest.mark.parametrize("nrhs", [3, 5, 12, 16, 19])
def test_hop_patch_parity(bq, L, prec, nrhs):
    import torch
    kappa = 0.125
    U = inputs.gauge(L, 71, 0.5)
    psis = rhs_set(L, nrhs, 72)
    recon = nrhs % 2
    for bc in (None, GENERAL_BC):
        with bq.Lattice(L, bc) as lat:
            bq.bq_gauge_load(lat.h, U)
            for p in (0, 1):
                src = import_multi(bq, lat, psis, prec, 1 - p)
                fb = bq.bq_field_bytes(lat.h, prec, p)
                out = torch.zeros(nrhs * fb, dtype=torch.uint8, device="cuda")
                bq.bq_wilson_apply_multi(lat.h, out, src, nrhs, kappa, p, prec, recon)
                got = export_multi(bq, lat, out, nrhs, prec, p)
                one = lat.field(prec, p)
                for k in range(nrhs):
                    ref = bqo.hop_restricted(U, psis[k], kappa, p, bc=bc)
                    assert relmax(got[k], ref) < TOL[prec], (L, prec, nrhs, k, p)
                    bq.bq_wilson_apply(lat.h, one, src[k * fb:(k + 1) * fb], kappa, p, prec, recon)
                    assert torch.equal(one, out[k * fb:(k + 1) * fb]), (L, prec, nrhs, k, p)


@pytest.mark.parametrize("inner,csw,method", [(1, 0.0, 0), (1, 1.0, 0), (2, 0.0, 0), (0, 1.0, 0), (1, 1.0, 1)])
def test_solve_multi_patch(bq, inner, csw, method):
    """Batched solve through the patch-mapped kernels (fused reductions, dagger hops for CGNR)."""
    L, kappa, nrhs = (16, 4, 4, 8), 0.1215, 6
    U = inputs.gauge(L, 73, 0.5)
    A = bqo.clover_build(U, csw, kappa) if csw else None
    b = np.stack(rhs_set(L, nrhs, 74))
    b[1] = 0
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        infos = bq.bq_solve_multi(lat.h, b, x, nrhs, kappa, 1e-10, bq.bq_solve_opts(inner_prec=inner, csw=csw, method=method))
    for k in range(nrhs):
        assert infos[k].status == 0
        if k == 1:
            assert not x[k].any()
        else:
            assert oracle_residual(U, x[k], b[k], kappa, A=A) <= 1e-10, k


def test_propagator_is_fig1_of_the_paper(bq):
    """bq_propagator = the loop of the paper's Fig. 1: 12 point sources at one site, one inversion each.
    Every column against the oracle's operator, and against the oracle's own BiCGStab solution."""
    L, kappa, csw = (4, 4, 4, 8), 0.12, 1.0
    U = inputs.gauge(L, 75, 0.4)
    A = bqo.clover_build(U, csw, kappa)
    src = (1, 2, 3, 5)
    S = np.full((12, L[3], L[2], L[1], L[0], 4, 3), np.nan, dtype=np.complex128)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        infos = bq.bq_propagator(lat.h, src, S, kappa, 1e-10, bq.bq_solve_opts(inner_prec=bq.BQ_FP32, csw=csw))
        with pytest.raises(bq.BqError):
            bq.bq_propagator(lat.h, (4, 0, 0, 0), S.copy(), kappa, 1e-10)
    assert len(infos) == 12 and all(i.status == 0 for i in infos)
    for s in range(4):
        for c in range(3):
            b = np.zeros(S.shape[1:], dtype=np.complex128)
            b[src[3], src[2], src[1], src[0], s, c] = 1.0
            k = 3 * s + c
            assert oracle_residual(U, S[k], b, kappa, A=A) <= 1e-10, k
            if k in (0, 7):
                x_ref, _ = bqo.bicgstab(U, b, kappa, tol=1e-12, A=A)
                assert np.linalg.norm(S[k] - x_ref) / np.linalg.norm(x_ref) < 1e-8


# ---------------------------------------------------------------------------------------------------
# link-stationary multi-rhs hop (hop_ls.cuh): links in registers for all right-hand sides of a 8 x 4 x 4 x 2 block of
# sites, spinor blocks + halos through shared memory by TMA.  Taken for fp32 / half storage when Lx % 16 == 0 and
# Ly % 4 == Lz % 4 == Lt % 2 == 0.  Lattices: one block in y, z, t (every halo wraps onto the block itself); several
# blocks per direction; three x tiles per row; wrap-around blocks in every direction with general boundary phases.
# ---------------------------------------------------------------------------------------------------
LS_LATTICES = [(16, 4, 4, 2), (16, 8, 4, 4), (32, 4, 8, 2), (48, 4, 4, 4)]


@pytest.mark.parametrize("L", LS_LATTICES)
@pytest.mark.parametrize("prec", [1, 2])
@pytest.mark.parametrize("nrhs", [2, 3, 12])
def test_hop_ls_parity(bq, L, prec, nrhs):
    import torch
    kappa = 0.125
    U = inputs.gauge(L, 81, 0.5)
    psis = rhs_set(L, nrhs, 82)
    recon = nrhs % 2
    for bc in (None, GENERAL_BC):
        with bq.Lattice(L, bc) as lat:
            bq.bq_gauge_load(lat.h, U)
            for p in (0, 1):
                src = import_multi(bq, lat, psis, prec, 1 - p)
                fb = bq.bq_field_bytes(lat.h, prec, p)
                out = torch.zeros(nrhs * fb, dtype=torch.uint8, device="cuda")
                n0 = bq.bq_get_counters(lat.h)["ls"]
                bq.bq_wilson_apply_multi(lat.h, out, src, nrhs, kappa, p, prec, recon)
                assert bq.bq_get_counters(lat.h)["ls"] == n0 + 1, "the link-stationary kernel did not take this launch"
                got = export_multi(bq, lat, out, nrhs, prec, p)
                one = lat.field(prec, p)
                for k in range(nrhs):
                    ref = bqo.hop_restricted(U, psis[k], kappa, p, bc=bc)
                    assert relmax(got[k], ref) < TOL[prec], (L, prec, nrhs, k, p)
                    bq.bq_wilson_apply(lat.h, one, src[k * fb:(k + 1) * fb], kappa, p, prec, recon)
                    assert torch.equal(one, out[k * fb:(k + 1) * fb]), (L, prec, nrhs, k, p)


@pytest.mark.parametrize("prec", [1, 2])
def test_ls_full_apply_and_schur(bq, prec):
    """[even | odd] buffers (operand stride = two fields), the xpay epilogue, and the Schur operator through the
    link-stationary kernel, every right-hand side against the oracle."""
    import torch
    L, kappa, nrhs = (16, 4, 8, 4), 0.12, 5
    U = inputs.gauge(L, 83, 0.4)
    psis = rhs_set(L, nrhs, 84)
    par = (inputs.site_parity(L) == 0)[..., None, None]
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        src = import_multi(bq, lat, psis, prec, bq.BQ_FULL)
        out = torch.zeros_like(src)
        n0 = bq.bq_get_counters(lat.h)["ls"]
        bq.bq_wilson_apply_multi(lat.h, out, src, nrhs, kappa, bq.BQ_FULL, prec, bq.BQ_RECON18)
        assert bq.bq_get_counters(lat.h)["ls"] == n0 + 2
        for k, got in enumerate(export_multi(bq, lat, out, nrhs, prec, bq.BQ_FULL)):
            assert relmax(got, bqo.dirac_apply(U, psis[k], kappa)) < TOL[prec], k
        src_e = import_multi(bq, lat, psis, prec, bq.BQ_EVEN)
        out_e, tmp = torch.zeros_like(src_e), torch.zeros_like(src_e)
        bq.bq_schur_apply_multi(lat.h, out_e, src_e, tmp, nrhs, kappa, 0.0, prec)
        assert bq.bq_get_counters(lat.h)["ls"] == n0 + 4
        for k, got in enumerate(export_multi(bq, lat, out_e, nrhs, prec, bq.BQ_EVEN)):
            ref = bqo.schur_apply(U, np.where(par, psis[k], 0), kappa)
            assert relmax(got, ref) < 2 * TOL[prec], (prec, k)


@pytest.mark.parametrize("inner,method", [(1, 0), (2, 0), (1, 1)])
def test_solve_multi_ls(bq, inner, method):
    """Batched Wilson solve whose inner hops all run through the link-stationary kernel (fused inner products, per-rhs
    done flags, dagger hops for CGNR); one zero and one tiny right-hand side stop early while the others go on."""
    L, kappa, nrhs = (16, 4, 4, 8), 0.1215, 6
    U = inputs.gauge(L, 85, 0.5)
    b = np.stack(rhs_set(L, nrhs, 86))
    b[1] = 0
    b[2] *= 1e-6
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        infos = bq.bq_solve_multi(lat.h, b, x, nrhs, kappa, 1e-10, bq.bq_solve_opts(inner_prec=inner, method=method, check_every=3))
        assert bq.bq_get_counters(lat.h)["ls"] > 0
        x1 = np.zeros_like(b[0])
        info1 = bq.bq_solve(lat.h, b[0], x1, kappa, 1e-10, bq.bq_solve_opts(inner_prec=inner, method=method, check_every=3))
    for k in range(nrhs):
        assert infos[k].status == 0
        if k == 1:
            assert not x[k].any()
        else:
            assert oracle_residual(U, x[k], b[k], kappa) <= 1e-10, k
    assert np.linalg.norm(x[0] - x1) / np.linalg.norm(x1) < 1e-9
    assert abs(infos[0].inner_iters - info1.inner_iters) <= 1      # the fused inner products are summed in another order


@pytest.mark.parametrize("prec", [1, 2])
def test_ls_clover_schur_and_solve(bq, prec):
    """Clover epilogues of the link-stationary kernel (clover tiles of the block in shared memory): the batched clover Schur
    operator against the oracle and against the single-field kernels bit for bit, then a batched clover solve."""
    import torch
    L, kappa, csw, nrhs = (16, 4, 8, 4), 0.1215, 1.0, 5
    U = inputs.gauge(L, 87, 0.5)
    psis = rhs_set(L, nrhs, 88)
    A = bqo.clover_build(U, csw, kappa)
    Ainv = bqo.site_matrix_invert(A)
    par = (inputs.site_parity(L) == 0)[..., None, None]
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        src = import_multi(bq, lat, psis, prec, bq.BQ_EVEN)
        out, tmp = torch.zeros_like(src), torch.zeros_like(src)
        n0 = bq.bq_get_counters(lat.h)["ls"]
        bq.bq_schur_apply_multi(lat.h, out, src, tmp, nrhs, kappa, csw, prec)
        assert bq.bq_get_counters(lat.h)["ls"] == n0 + 2, "the clover hops did not take the link-stationary kernel"
        fb = bq.bq_field_bytes(lat.h, prec, bq.BQ_EVEN)
        one, tmp1 = lat.field(prec, bq.BQ_EVEN), lat.field(prec, bq.BQ_EVEN)
        for k, got in enumerate(export_multi(bq, lat, out, nrhs, prec, bq.BQ_EVEN)):
            ref = bqo.schur_apply(U, np.where(par, psis[k], 0), kappa, A=A, Ainv=Ainv)
            assert relmax(got, ref) < 2 * TOL[prec], (prec, k)
            bq.bq_schur_apply(lat.h, one, src[k * fb:(k + 1) * fb], tmp1, kappa, csw, prec)
            assert torch.equal(one, out[k * fb:(k + 1) * fb]), (prec, k)
        b = np.stack(psis)
        b[1] = 0
        x = np.zeros_like(b)
        n0 = bq.bq_get_counters(lat.h)["ls"]
        infos = bq.bq_solve_multi(lat.h, b, x, nrhs, kappa, 1e-10, bq.bq_solve_opts(inner_prec=prec, csw=csw, check_every=3))
        assert bq.bq_get_counters(lat.h)["ls"] > n0
    for k in range(nrhs):
        assert infos[k].status == 0
        if k != 1:
            assert oracle_residual(U, x[k], b[k], kappa, A=A) <= 1e-10, k


# ---------------------------------------------------------------------------------------------------
# Direction-split pipelined link-stationary kernel (hop_lsp.cuh): two threads per site, four directions each, the
# accumulator handed over through shared memory in the order of the single-rhs kernel — so the results must again be bit
# for bit those of hop_kernel.  By default it serves fp64 with >= 8 right-hand sides; BQ_MRHS_LS=3 (read when the handle
# is created) sends every eligible launch through it.
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", LS_LATTICES)
@pytest.mark.parametrize("prec", [0, 1, 2])
@pytest.mark.parametrize("nrhs", [2, 3, 12])
def test_hop_lsp_parity(bq, L, prec, nrhs, monkeypatch):
    import torch
    monkeypatch.setenv("BQ_MRHS_LS", "3")
    kappa = 0.125
    U = inputs.gauge(L, 91, 0.5)
    psis = rhs_set(L, nrhs, 92)
    recon = nrhs % 2
    for bc in (None, GENERAL_BC):
        with bq.Lattice(L, bc) as lat:
            bq.bq_gauge_load(lat.h, U)
            for p in (0, 1):
                src = import_multi(bq, lat, psis, prec, 1 - p)
                fb = bq.bq_field_bytes(lat.h, prec, p)
                out = torch.zeros(nrhs * fb, dtype=torch.uint8, device="cuda")
                n0 = bq.bq_get_counters(lat.h)["lsp"]
                bq.bq_wilson_apply_multi(lat.h, out, src, nrhs, kappa, p, prec, recon)
                assert bq.bq_get_counters(lat.h)["lsp"] == n0 + 1, "the direction-split kernel did not take this launch"
                got = export_multi(bq, lat, out, nrhs, prec, p)
                one = lat.field(prec, p)
                for k in range(nrhs):
                    ref = bqo.hop_restricted(U, psis[k], kappa, p, bc=bc)
                    assert relmax(got[k], ref) < TOL[prec], (L, prec, nrhs, k, p)
                    bq.bq_wilson_apply(lat.h, one, src[k * fb:(k + 1) * fb], kappa, p, prec, recon)
                    assert torch.equal(one, out[k * fb:(k + 1) * fb]), (L, prec, nrhs, k, p)


@pytest.mark.parametrize("prec", [0, 1, 2])
def test_lsp_full_apply_schur_and_dagger(bq, prec, monkeypatch):
    """[even | odd] buffers (operand stride = two fields), the xpay epilogue, the Schur operator and the dagger modes through
    the direction-split kernel, every right-hand side against the oracle."""
    import torch
    monkeypatch.setenv("BQ_MRHS_LS", "3")
    L, kappa, nrhs = (16, 4, 8, 4), 0.12, 5
    U = inputs.gauge(L, 93, 0.4)
    psis = rhs_set(L, nrhs, 94)
    par = (inputs.site_parity(L) == 0)[..., None, None]
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        src = import_multi(bq, lat, psis, prec, bq.BQ_FULL)
        out = torch.zeros_like(src)
        n0 = bq.bq_get_counters(lat.h)["lsp"]
        bq.bq_wilson_apply_multi(lat.h, out, src, nrhs, kappa, bq.BQ_FULL, prec, bq.BQ_RECON18)
        assert bq.bq_get_counters(lat.h)["lsp"] == n0 + 2
        for k, got in enumerate(export_multi(bq, lat, out, nrhs, prec, bq.BQ_FULL)):
            assert relmax(got, bqo.dirac_apply(U, psis[k], kappa)) < TOL[prec], k
        src_e = import_multi(bq, lat, psis, prec, bq.BQ_EVEN)
        out_e, tmp = torch.zeros_like(src_e), torch.zeros_like(src_e)
        bq.bq_schur_apply_multi(lat.h, out_e, src_e, tmp, nrhs, kappa, 0.0, prec)
        assert bq.bq_get_counters(lat.h)["lsp"] == n0 + 4
        for k, got in enumerate(export_multi(bq, lat, out_e, nrhs, prec, bq.BQ_EVEN)):
            ref = bqo.schur_apply(U, np.where(par, psis[k], 0), kappa)
            assert relmax(got, ref) < 2 * TOL[prec], (prec, k)


@pytest.mark.parametrize("inner,method", [(1, 0), (2, 0), (1, 1), (0, 0)])
def test_solve_multi_lsp(bq, inner, method, monkeypatch):
    """Batched Wilson solve whose hops all run through the direction-split kernel (fused inner products in role B, per-rhs done
    flags, dagger hops for CGNR, fp64 outer residuals); one zero and one tiny right-hand side stop early."""
    monkeypatch.setenv("BQ_MRHS_LS", "3")
    L, kappa, nrhs = (16, 4, 4, 8), 0.1215, 6
    U = inputs.gauge(L, 95, 0.5)
    b = np.stack(rhs_set(L, nrhs, 96))
    b[1] = 0
    b[2] *= 1e-6
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        infos = bq.bq_solve_multi(lat.h, b, x, nrhs, kappa, 1e-10, bq.bq_solve_opts(inner_prec=inner, method=method, check_every=3))
        assert bq.bq_get_counters(lat.h)["lsp"] > 0
        x1 = np.zeros_like(b[0])
        info1 = bq.bq_solve(lat.h, b[0], x1, kappa, 1e-10, bq.bq_solve_opts(inner_prec=inner, method=method, check_every=3))
    for k in range(nrhs):
        assert infos[k].status == 0
        if k == 1:
            assert not x[k].any()
        else:
            assert oracle_residual(U, x[k], b[k], kappa) <= 1e-10, k
    assert np.linalg.norm(x[0] - x1) / np.linalg.norm(x1) < 1e-9
    assert abs(infos[0].inner_iters - info1.inner_iters) <= 1      # the fused inner products are summed in another order


def test_lsp_is_the_default_for_fp64_batches(bq):
    """Without the switch: fp64 with >= 8 right-hand sides takes the direction-split kernel, fp32 the one-thread-per-site one."""
    import torch
    L, kappa, nrhs = (16, 4, 4, 4), 0.125, 8
    U = inputs.gauge(L, 97, 0.5)
    psis = rhs_set(L, nrhs, 98)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        for prec, want in ((0, 1), (1, 0)):
            src = import_multi(bq, lat, psis, prec, 1)
            out = torch.zeros_like(src)
            c0 = bq.bq_get_counters(lat.h)
            bq.bq_wilson_apply_multi(lat.h, out, src, nrhs, kappa, 0, prec, bq.BQ_RECON18)
            c1 = bq.bq_get_counters(lat.h)
            assert c1["ls"] == c0["ls"] + 1 and c1["lsp"] == c0["lsp"] + want, (prec, c0, c1)
            for k, got in enumerate(export_multi(bq, lat, out, nrhs, prec, 0)):
                assert relmax(got, bqo.hop_restricted(U, psis[k], kappa, 0)) < TOL[prec], (prec, k)


@pytest.mark.parametrize("nrhs", [16, 19])
def test_lsp_fp64_full_and_chunked_batches(bq, nrhs):
    """fp64, default kernel choice: 16 right-hand sides (the most one launch holds) and 19 (two chunks of 10 + 9, both >= 8) go through the
    direction-split kernel; every right-hand side against the oracle and bit for bit against the single-rhs kernel."""
    import torch
    L, kappa = (16, 4, 8, 2), 0.125
    U = inputs.gauge(L, 101, 0.5)
    psis = rhs_set(L, nrhs, 102)
    with bq.Lattice(L, GENERAL_BC) as lat:
        bq.bq_gauge_load(lat.h, U)
        src = import_multi(bq, lat, psis, 0, 1)
        fb = bq.bq_field_bytes(lat.h, 0, 0)
        out = torch.zeros(nrhs * fb, dtype=torch.uint8, device="cuda")
        c0 = bq.bq_get_counters(lat.h)
        bq.bq_wilson_apply_multi(lat.h, out, src, nrhs, kappa, 0, 0, bq.BQ_RECON18)
        c1 = bq.bq_get_counters(lat.h)
        nlaunch = (nrhs + 15) // 16
        assert c1["lsp"] == c0["lsp"] + nlaunch and c1["ls"] == c0["ls"] + nlaunch
        one = lat.field(0, 0)
        for k, got in enumerate(export_multi(bq, lat, out, nrhs, 0, 0)):
            assert relmax(got, bqo.hop_restricted(U, psis[k], kappa, 0, bc=GENERAL_BC)) < TOL[0], k
            bq.bq_wilson_apply(lat.h, one, src[k * fb:(k + 1) * fb], kappa, 0, 0, bq.BQ_RECON18)
            assert torch.equal(one, out[k * fb:(k + 1) * fb]), k
