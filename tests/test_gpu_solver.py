"""GPU parity for the fused BLAS-1 kernels (A6) and bq_solve (A7-A10) against numpy / the CPU oracle.

Solves: any x with true residual |b - D x|/|b| <= tol is correct; the residual is recomputed
here with the ORACLE's operator, never trusted from the library.  Iteration counts are reported, not matched.
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


def even_part(L, psi):
    return np.where((inputs.site_parity(L) == 0)[..., None, None], psi, 0)


# storage rounding of the operands, then sums of ~N products: tolerances relative to |a||b|
BLAS_TOL = {0: 1e-13, 1: 2e-6, 2: 2e-3}


@pytest.mark.parametrize("prec", [0, 1, 2])
@pytest.mark.parametrize("L", [(4, 4, 4, 4), (8, 6, 6, 10)])
def test_blas_reductions_and_axpy(bq, prec, L):
    a = even_part(L, inputs.spinor(L, 41))
    b = even_part(L, inputs.spinor(L, 42, inputs.STREAM_TEST))
    with bq.Lattice(L) as lat:
        da, db = lat.import_field(a, prec, bq.BQ_EVEN), lat.import_field(b, prec, bq.BQ_EVEN)
        # compare against numpy on the values as stored (export = exact view of the stored numbers)
        sa, sb = lat.export_field(da, prec, bq.BQ_EVEN), lat.export_field(db, prec, bq.BQ_EVEN)
        n2 = bq.bq_blas_norm2(lat.h, da, prec)
        assert abs(n2 - np.vdot(sa, sa).real) <= 1e-6 * n2 if prec else abs(n2 - np.vdot(sa, sa).real) <= 1e-13 * n2
        assert abs(n2 - np.vdot(a, a).real) <= 2 * BLAS_TOL[prec] * n2 + 1e-13 * n2
        dot = bq.bq_blas_cdot(lat.h, da, db, prec)
        scale = np.linalg.norm(a) * np.linalg.norm(b)
        assert abs(dot - np.vdot(sa, sb)) <= (1e-6 if prec else 1e-13) * scale
        assert abs(dot - np.vdot(a, b)) <= BLAS_TOL[prec] * scale
        # bitwise reproducible reductions
        assert bq.bq_blas_cdot(lat.h, da, db, prec) == dot and bq.bq_blas_norm2(lat.h, da, prec) == n2
        alpha = 0.3 - 0.7j
        bq.bq_blas_caxpy(lat.h, alpha, da, db, prec)
        got = lat.export_field(db, prec, bq.BQ_EVEN)
        ref = sb + alpha * sa
        tol = {0: 1e-15, 1: 3e-7, 2: 1e-3}[prec]
        assert np.abs(got - ref).max() <= tol * np.abs(ref).max()


@pytest.mark.parametrize("prec", [0, 1, 2])
def test_blas_bicg_update(bq, prec):
    L = (8, 4, 4, 6)
    vec = [even_part(L, inputs.spinor(L, 50 + k)) for k in range(6)]
    alpha, omega = 0.8 + 0.1j, 0.6 - 0.2j
    with bq.Lattice(L) as lat:
        xprec = bq.BQ_FP32 if prec == bq.BQ_HALF else prec
        p, s, t, rhat, r = [lat.import_field(v, prec, bq.BQ_EVEN) for v in vec[:5]]
        x = lat.import_field(vec[5], xprec, bq.BQ_EVEN)
        sp, ss, st, srhat = [lat.export_field(d, prec, bq.BQ_EVEN) for d in (p, s, t, rhat)]
        sx = lat.export_field(x, xprec, bq.BQ_EVEN)
        r2, rr = bq.bq_blas_bicg_update(lat.h, alpha, omega, p, s, t, rhat, x, r, prec)
        x_ref = sx + alpha * sp + omega * ss
        r_ref = ss - omega * st
        tol = {0: 1e-15, 1: 5e-7, 2: 1e-3}[prec]
        assert np.abs(lat.export_field(x, xprec, bq.BQ_EVEN) - x_ref).max() <= (5e-7 if prec else 1e-15) * np.abs(x_ref).max()
        got_r = lat.export_field(r, prec, bq.BQ_EVEN)
        assert np.abs(got_r - r_ref).max() <= tol * np.abs(r_ref).max()
        rtol = {0: 1e-13, 1: 1e-6, 2: 1e-6}[prec]     # reductions are over r as stored
        assert abs(r2 - np.vdot(got_r, got_r).real) <= rtol * r2
        assert abs(rr - np.vdot(srhat, got_r)) <= rtol * np.linalg.norm(srhat) * np.linalg.norm(got_r)


# ---------------------------------------------------------------------------------------------------
# solves
# ---------------------------------------------------------------------------------------------------
def oracle_residual(U, x, b, kappa, A=None):
    return np.linalg.norm(b - bqo.dirac_apply(U, x, kappa, A=A)) / np.linalg.norm(b)


def test_config1_solve_fp64(bq, cfg1):
    """BASELINE.json config 1: 4^4 fp64 BiCGStab to 1e-12."""
    U, b, kappa, L = cfg1["U"], cfg1["b"], cfg1["kappa"], cfg1["L"]
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        opts = bq.bq_solve_opts(inner_prec=bq.BQ_FP64)
        info = bq.bq_solve(lat.h, b, x, kappa, 1e-12, opts)
    assert info.status == 0 and info.true_rel_residual <= 1e-12
    assert oracle_residual(U, x, b, kappa) <= 1e-12
    x_ref, oinfo = bqo.bicgstab(U, b, kappa, tol=1e-13)
    assert np.linalg.norm(x - x_ref) / np.linalg.norm(x_ref) < 1e-10
    assert 0 < info.inner_iters < 200
    print("config1 fp64: iters", info.inner_iters, "restarts", info.restarts, "oracle iters (full D)", oinfo["iters"])


@pytest.mark.parametrize("inner,recon", [(1, 0), (1, 1), (2, 0), (2, 1)])
def test_mixed_precision_wilson_solve(bq, inner, recon):
    L = (8, 8, 8, 8)
    kappa = 0.1235
    U = inputs.gauge(L, 61, 0.7)
    b = inputs.spinor(L, 61)
    import torch
    xd = torch.zeros(b.shape, dtype=torch.complex128, device="cuda")     # device-resident b and x
    bd = torch.from_numpy(b).cuda()
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        opts = bq.bq_solve_opts(inner_prec=inner, recon=recon)
        info = bq.bq_solve(lat.h, bd, xd, kappa, 1e-10, opts)
    x = xd.cpu().numpy()
    res = oracle_residual(U, x, b, kappa)
    print(f"inner={inner} recon={recon}: outer {info.outer_cycles} inner iters {info.inner_iters} true res {res:.2e}")
    assert info.status == 0 and res <= 1e-10 and abs(res - info.true_rel_residual) < 1e-11
    assert info.outer_cycles >= 2


@pytest.mark.parametrize("inner", [0, 1, 2])
def test_clover_solve(bq, inner):
    L = (8, 4, 8, 8)
    csw, kappa = 1.0, 0.1215
    U = inputs.gauge(L, 62, 0.5)
    b = inputs.spinor(L, 62)
    A = bqo.clover_build(U, csw, kappa)
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        opts = bq.bq_solve_opts(inner_prec=inner, csw=csw)
        info = bq.bq_solve(lat.h, b, x, kappa, 1e-10, opts)
    res = oracle_residual(U, x, b, kappa, A=A)
    print(f"clover inner={inner}: outer {info.outer_cycles} iters {info.inner_iters} res {res:.2e}")
    assert info.status == 0 and res <= 1e-10
    x_ref, _ = bqo.bicgstab(U, b, kappa, tol=1e-12, A=A)
    assert np.linalg.norm(x - x_ref) / np.linalg.norm(x_ref) < 1e-8


def test_solve_with_initial_guess_and_zero_rhs(bq, cfg1):
    U, b, kappa, L = cfg1["U"], cfg1["b"], cfg1["kappa"], cfg1["L"]
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        x = np.zeros_like(b)
        info0 = bq.bq_solve(lat.h, b, x, kappa, 1e-10)
        x1 = x.copy()
        info1 = bq.bq_solve(lat.h, b, x1, kappa, 1e-10)             # start from the solution: nothing to do
        assert info1.inner_iters == 0 and np.array_equal(np.isfinite(x1), np.ones_like(x1, dtype=bool))
        assert oracle_residual(U, x1, b, kappa) <= 1e-10
        xz = inputs.spinor(L, 5)
        infoz = bq.bq_solve(lat.h, np.zeros_like(b), xz, kappa, 1e-10)
        assert infoz.status == 0 and np.all(xz == 0)
        assert info0.inner_iters > 0


def test_solve_reports_non_convergence(bq, cfg1):
    U, b, kappa, L = cfg1["U"], cfg1["b"], cfg1["kappa"], cfg1["L"]
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        x = np.zeros_like(b)
        opts = bq.bq_solve_opts(inner_prec=bq.BQ_FP32, max_inner=2, max_outer=2, check_every=1)
        info = bq.bq_solve(lat.h, b, x, kappa, 1e-12, opts, raise_on_fail=False)
        assert info.status == bq.BQ_ENOTCONVERGED
        # x holds the best iterate and the reported residual is the true one
        assert abs(oracle_residual(U, x, b, kappa) - info.true_rel_residual) < 1e-9
        with pytest.raises(bq.BqError):
            bq.bq_solve(lat.h, b, x, kappa, -1.0)


@pytest.mark.parametrize("inner", [0, 1, 2])
@pytest.mark.parametrize("csw", [0.0, 1.0])
def test_lexical_solve(bq, inner, csw):
    """BiCGStab on the full matrix D (no even-odd preconditioning) — the oracle's own formulation."""
    L, kappa = (8, 4, 8, 8), 0.1215
    U = inputs.gauge(L, 63, 0.5)
    b = inputs.spinor(L, 63)
    A = bqo.clover_build(U, csw, kappa) if csw else None
    x, xe = np.zeros_like(b), np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        info = bq.bq_solve(lat.h, b, x, kappa, 1e-10, bq.bq_solve_opts(inner_prec=inner, csw=csw, lexical=1))
        info_eo = bq.bq_solve(lat.h, b, xe, kappa, 1e-10, bq.bq_solve_opts(inner_prec=inner, csw=csw))
        with pytest.raises(bq.BqError):
            bq.bq_solve(lat.h, b, x.copy(), kappa, 1e-10, bq.bq_solve_opts(lexical=1, method=bq.BQ_CGNR))
        xz = inputs.spinor(L, 5)
        infoz = bq.bq_solve(lat.h, np.zeros_like(b), xz, kappa, 1e-10, bq.bq_solve_opts(lexical=1))
        assert infoz.status == 0 and np.all(xz == 0)
    res = oracle_residual(U, x, b, kappa, A=A)
    _, oinfo = bqo.bicgstab(U, b, kappa, tol=1e-10, A=A)
    print(f"lexical inner={inner} csw={csw}: outer {info.outer_cycles} iters {info.inner_iters} (even-odd {info_eo.inner_iters}, "
          f"oracle on full D {oinfo['iters']}) res {res:.2e}")
    assert info.status == 0 and res <= 1e-10 and abs(res - info.true_rel_residual) < 1e-11
    assert np.linalg.norm(x - xe) / np.linalg.norm(xe) < 1e-8
    assert info.inner_iters > info_eo.inner_iters          # preconditioning helps (cond M^ < cond D)


def test_solve_x0_zero_ignores_x_on_entry(bq, cfg1):
    """opts.x0_zero: x is output only — NaN garbage on entry must not matter, and the result equals the zero-guess solve."""
    U, b, kappa, L = cfg1["U"], cfg1["b"], cfg1["kappa"], cfg1["L"]
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        x_ref = np.zeros_like(b)
        bq.bq_solve(lat.h, b, x_ref, kappa, 1e-10)
        x = np.full_like(b, np.nan)
        info = bq.bq_solve(lat.h, b, x, kappa, 1e-10, bq.bq_solve_opts(inner_prec=bq.BQ_FP32, x0_zero=1))
        assert info.status == 0 and np.array_equal(x, x_ref)
        xm = np.full((2,) + b.shape, np.nan, dtype=np.complex128)
        infos = bq.bq_solve_multi(lat.h, np.stack([b, 2 * b]), xm, 2, kappa, 1e-10, bq.bq_solve_opts(inner_prec=bq.BQ_FP32, x0_zero=1))
        assert all(i.status == 0 for i in infos)
        assert oracle_residual(U, xm[0], b, kappa) <= 1e-10 and oracle_residual(U, xm[1], 2 * b, kappa) <= 1e-10


def test_graph_replay_matches_eager_and_survives_reconfiguration(bq, monkeypatch):
    """The batches of inner iterations are replayed as CUDA graphs from their third occurrence on (eager, capture, replay).
    The solution must be bitwise that of eager launches (BQ_GRAPH=0), and a cached graph must not outlive what it points
    at: another batch shape, another precision, a multi-rhs solve in between (reduction scratch regrows), a new gauge field."""
    L, kappa = (8, 8, 8, 8), 0.124
    U, U2 = inputs.gauge(L, 81, 0.6), inputs.gauge(L, 82, 0.6)
    b = inputs.spinor(L, 81)
    opts = bq.bq_solve_opts(inner_prec=bq.BQ_FP32, check_every=2, x0_zero=1)       # many full batches per solve

    def solve(lat, rhs=b, o=opts):
        x = np.empty_like(rhs)
        info = bq.bq_solve(lat.h, rhs, x, kappa, 1e-10, o)
        return x, info

    monkeypatch.setenv("BQ_GRAPH", "0")
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        x_eager, info_eager = solve(lat)
        c_eager = bq.bq_get_counters(lat.h)
        bq.bq_gauge_load(lat.h, U2)
        x2_eager, _ = solve(lat)
    monkeypatch.setenv("BQ_GRAPH", "1")
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        x1, info1 = solve(lat)
        c1 = bq.bq_get_counters(lat.h)
        assert np.array_equal(x1, x_eager) and info1.inner_iters == info_eager.inner_iters
        assert c1 == c_eager                                   # replays are counted like the launches they stand for
        for _ in range(3):
            x, _ = solve(lat)
            assert np.array_equal(x, x_eager)
        xh, ih = solve(lat, o=bq.bq_solve_opts(inner_prec=bq.BQ_HALF, check_every=2, x0_zero=1))
        assert ih.status == 0 and oracle_residual(U, xh, b, kappa) <= 1e-10
        xm = np.empty((3,) + b.shape, dtype=np.complex128)
        infos = bq.bq_solve_multi(lat.h, np.stack([b, 2 * b, -b]), xm, 3, kappa, 1e-10, opts)
        assert all(i.status == 0 for i in infos) and oracle_residual(U, xm[2], -b, kappa) <= 1e-10
        x, _ = solve(lat)
        assert np.array_equal(x, x_eager)
        xc, ic = solve(lat, o=bq.bq_solve_opts(inner_prec=bq.BQ_FP32, check_every=2, x0_zero=1, method=bq.BQ_CGNR))
        assert ic.status == 0 and oracle_residual(U, xc, b, kappa) <= 1e-10
        bq.bq_gauge_load(lat.h, U2)
        x2, _ = solve(lat)
        assert np.array_equal(x2, x2_eager) and oracle_residual(U2, x2, b, kappa) <= 1e-10


@pytest.mark.parametrize("inner,method", [(1, 0), (2, 0), (0, 0), (1, 1)])
def test_near_free_field_long_solve(bq, inner, method):
    """A smooth field (eps = 0.05) close to the free critical point (kappa = 0.1245): ~90 iterations instead of ~12, i.e.
    many batches (graph replays), several half-precision outer cycles — all judged with the oracle's operator."""
    L, kappa = (8, 8, 8, 16), 0.1245
    U = inputs.gauge(L, 777, 0.05)
    b = inputs.spinor(L, 777)
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        info = bq.bq_solve(lat.h, b, x, kappa, 1e-10, bq.bq_solve_opts(inner_prec=inner, method=method, max_inner=2000, max_outer=100))
    res = oracle_residual(U, x, b, kappa)
    print(f"near-free inner={inner} method={method}: outer {info.outer_cycles} iters {info.inner_iters} res {res:.2e}")
    assert info.status == 0 and res <= 1e-10 and abs(res - info.true_rel_residual) < 1e-11
    assert info.inner_iters > 40


def test_nan_rhs_is_rejected(bq):
    """A right-hand side with a NaN must not come back as BQ_OK with x = x0 (|b| = NaN compares false with everything)."""
    L, kappa = (4, 4, 4, 4), 0.12
    U = inputs.gauge(L, 901, 0.3)
    b = inputs.spinor(L, 902)
    b[1, 2, 3, 0, 1, 2] = np.nan
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        for o in (None, bq.bq_solve_opts(inner_prec=bq.BQ_FP64), bq.bq_solve_opts(inner_prec=bq.BQ_FP32, lexical=1)):
            with pytest.raises(bq.BqError) as e:
                bq.bq_solve(lat.h, b, x, kappa, 1e-10, o)
            assert e.value.status == bq.BQ_EINVAL
        bb = np.stack([inputs.spinor(L, 903), b])
        with pytest.raises(bq.BqError) as e:
            bq.bq_solve_multi(lat.h, bb, np.zeros_like(bb), 2, kappa, 1e-10)
        assert e.value.status == bq.BQ_EINVAL
        # the handle is still usable
        b2 = inputs.spinor(L, 904)
        info = bq.bq_solve(lat.h, b2, x, kappa, 1e-10)
        assert info.status == 0 and oracle_residual(U, x, b2, kappa) <= 1e-10


def test_batch_statuses_are_per_rhs(bq):
    """bq_solve_multi: every right-hand side stops on its own criterion and gets its own status (include/bq.h): with an
    iteration budget too small for the Gaussian sources, the zero right-hand side is still BQ_OK, the others are
    BQ_ENOTCONVERGED, and the call returns the failure."""
    L, kappa, nrhs = (8, 4, 4, 8), 0.1215, 3
    U = inputs.gauge(L, 905, 0.5)
    b = np.stack([inputs.spinor(L, 906 + k) for k in range(nrhs)])
    b[1] = 0
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        opts = bq.bq_solve_opts(inner_prec=bq.BQ_FP32, max_inner=2, max_outer=2, check_every=1)
        with pytest.raises(bq.BqError) as e:
            bq.bq_solve_multi(lat.h, b, x, nrhs, kappa, 1e-12, opts)
        assert e.value.status == bq.BQ_ENOTCONVERGED
        infos = bq.bq_solve_multi(lat.h, b, x, nrhs, kappa, 1e-12, opts, raise_on_fail=False)
        assert [i.status for i in infos] == [bq.BQ_ENOTCONVERGED, bq.BQ_OK, bq.BQ_ENOTCONVERGED]
        assert not x[1].any() and infos[1].inner_iters == 0
        # and with a normal budget every one converges
        infos = bq.bq_solve_multi(lat.h, b, x, nrhs, kappa, 1e-10, bq.bq_solve_opts(inner_prec=bq.BQ_FP32))
        assert all(i.status == 0 for i in infos)
        for k in (0, 2):
            assert oracle_residual(U, x[k], b[k], kappa) <= 1e-10


def test_binding_rejects_wrong_arrays(bq):
    """The binding checks what the C side cannot see: dtype, contiguity, element count (it never copies or converts)."""
    L, kappa = (4, 4, 4, 4), 0.12
    U = inputs.gauge(L, 911, 0.3)
    b = inputs.spinor(L, 912)
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        for bad_b, bad_x in ((b.astype(np.complex64), x), (b, x[..., ::-1]), (b[:2], x), (b, np.zeros((2,) + b.shape, dtype=np.complex128))):
            with pytest.raises(bq.BqError) as e:
                bq.bq_solve(lat.h, bad_b, bad_x, kappa, 1e-10)
            assert e.value.status == bq.BQ_EINVAL
        with pytest.raises(bq.BqError):
            bq.bq_solve_multi(lat.h, np.stack([b, b]), np.zeros((3,) + b.shape, dtype=np.complex128), 2, kappa, 1e-10)


def test_clover_apply_in_place_and_on_a_stream(bq):
    """bq_clover_apply: out may equal in (include/bq.h), and the apply runs on the caller's stream."""
    import torch
    L, kappa, csw = (4, 4, 6, 4), 0.12, 1.0
    U = inputs.gauge(L, 913, 0.5)
    psi = inputs.spinor(L, 914)
    A = bqo.clover_build(U, csw, kappa)
    ref = bqo.site_matrix_apply(A, psi)
    st = torch.cuda.Stream()
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        for prec, tol in ((bq.BQ_FP64, 1e-12), (bq.BQ_FP32, 1e-5)):
            buf = lat.import_field(psi, prec, bq.BQ_FULL)
            out = torch.zeros_like(buf)
            bq.bq_clover_apply(lat.h, csw, kappa, out, buf, bq.BQ_FULL, 0, prec, st)
            st.synchronize()
            bq.bq_clover_apply(lat.h, csw, kappa, buf, buf, bq.BQ_FULL, 0, prec)       # in place
            torch.cuda.synchronize()
            assert torch.equal(out, buf)
            assert relmax(lat.export_field(buf, prec, bq.BQ_FULL), ref) < tol
