"""GPU parity of the operator modes D, Ddag, DdagD (PAPER.md:44 set_mode) against the oracle's
adjoint (oracle/bqo.c bqo_dirac_apply_dag: the definition of the adjoint, pinned in tests/test_oracle_dagger_pins.py)."""
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


@pytest.mark.parametrize("L", [(8, 4, 6, 4), (6, 6, 4, 10), (4, 2, 6, 2)])
@pytest.mark.parametrize("prec", [0, 1, 2])
@pytest.mark.parametrize("csw", [0.0, 1.0])
def test_dirac_modes(bq, L, prec, csw):
    kappa = 0.1215
    U = inputs.gauge(L, 91, 0.5)
    psi = inputs.spinor(L, 91)
    A = bqo.clover_build(U, csw, kappa) if csw else None
    recon = 1 if prec == 1 else 0
    for bc in (None, GENERAL_BC):
        d = bqo.dirac_apply(U, psi, kappa, bc=bc, A=A)
        ref = {bq.BQ_MODE_D: d, bq.BQ_MODE_DDAG: bqo.dirac_apply_dag(U, psi, kappa, bc=bc, A=A),
               bq.BQ_MODE_DDAGD: bqo.dirac_apply_dag(U, d, kappa, bc=bc, A=A)}
        with bq.Lattice(L, bc) as lat:
            bq.bq_gauge_load(lat.h, U)
            src = lat.import_field(psi, prec, bq.BQ_FULL)
            out, tmp = lat.field(prec, bq.BQ_FULL), lat.field(prec, bq.BQ_FULL)
            for mode, r in ref.items():
                bq.bq_dirac_apply_mode(lat.h, out, src, tmp, kappa, csw, mode, prec, recon)
                got = lat.export_field(out, prec, bq.BQ_FULL)
                assert relmax(got, r) < (2 if mode == bq.BQ_MODE_DDAGD else 1) * TOL[prec], (L, prec, csw, mode)
            with pytest.raises(bq.BqError):
                bq.bq_dirac_apply_mode(lat.h, out, src, None, kappa, csw, bq.BQ_MODE_DDAGD, prec, recon)


@pytest.mark.parametrize("prec", [0, 1, 2])
@pytest.mark.parametrize("csw", [0.0, 1.0])
def test_schur_modes(bq, prec, csw):
    """M^^dag from the oracle: masked full-lattice applies of D^dag (the same Schur algebra as bqo.schur_apply)."""
    L, kappa = (8, 4, 6, 4), 0.1215
    U = inputs.gauge(L, 92, 0.5)
    psi = inputs.spinor(L, 92)
    A = bqo.clover_build(U, csw, kappa) if csw else None
    Ainv = bqo.site_matrix_invert(A) if csw else None
    even = (inputs.site_parity(L) == 0)[..., None, None]

    def schur_dag(v):
        xe = np.where(even, v, 0)
        y = bqo.dirac_apply_dag(U, xe, kappa, A=A)         # even: A_ee x_e ; odd: -kappa H^dag_oe x_e
        y_o = np.where(~even, y, 0)
        if Ainv is not None:
            y_o = bqo.site_matrix_apply(Ainv, y_o)
        z = bqo.dirac_apply_dag(U, y_o, kappa, A=A)
        return np.where(even, y, 0) - np.where(even, z, 0)

    m = bqo.schur_apply(U, np.where(even, psi, 0), kappa, A=A, Ainv=Ainv)
    ref = {bq.BQ_MODE_D: m, bq.BQ_MODE_DDAG: schur_dag(psi), bq.BQ_MODE_DDAGD: schur_dag(m)}
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        xe = lat.import_field(psi, prec, bq.BQ_EVEN)
        out, t1, t2 = (lat.field(prec, bq.BQ_EVEN) for _ in range(3))
        for mode, r in ref.items():
            bq.bq_schur_apply_mode(lat.h, out, xe, t1, t2, kappa, csw, mode, prec)
            assert relmax(lat.export_field(out, prec, bq.BQ_EVEN), r) < (4 if mode == bq.BQ_MODE_DDAGD else 2) * TOL[prec], (prec, csw, mode)


def test_dagger_adjointness_full_size(bq):
    """32^3 x 64 (BASELINE config 3 shape), fp64: <x, D y> = <D^dag x, y> with both sides from the GPU and the oracle's
    D y on sampled sites as the anchor for D."""
    import torch
    L, kappa = (32, 32, 32, 64), 0.125
    U = inputs.gauge(L, inputs.BASE_SEED + 3, 0.5)
    x, y = inputs.spinor(L, 93), inputs.spinor(L, 94, inputs.STREAM_TEST)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        dx, dy = lat.import_field(x, 0, bq.BQ_FULL), lat.import_field(y, 0, bq.BQ_FULL)
        out = lat.field(0, bq.BQ_FULL)
        bq.bq_dirac_apply_mode(lat.h, out, dy, None, kappa, 0.0, bq.BQ_MODE_D, 0)
        Dy = lat.export_field(out, 0, bq.BQ_FULL)
        bq.bq_dirac_apply_mode(lat.h, out, dx, None, kappa, 0.0, bq.BQ_MODE_DDAG, 0)
        Ddx = lat.export_field(out, 0, bq.BQ_FULL)
    sites = np.random.default_rng(5).integers(0, x.size // 12, 4096)
    assert relmax(Dy.reshape(-1, 4, 3)[sites], bqo.dirac_apply_sites(U, y, kappa, sites)) < 1e-12
    lhs, rhs = np.vdot(x, Dy), np.vdot(Ddx, y)
    assert abs(lhs - rhs) / abs(lhs) < 1e-12


# ---------------------------------------------------------------------------------------------------
# CG on the normal equations (bq_solve_opts.method = BQ_CGNR), judged with the ORACLE's operator
# ---------------------------------------------------------------------------------------------------
def oracle_residual(U, x, b, kappa, A=None):
    return np.linalg.norm(b - bqo.dirac_apply(U, x, kappa, A=A)) / np.linalg.norm(b)


@pytest.mark.parametrize("inner", [0, 1, 2])
@pytest.mark.parametrize("csw", [0.0, 1.0])
def test_cgnr_solve(bq, inner, csw):
    L, kappa = (8, 4, 8, 8), 0.1215
    U = inputs.gauge(L, 95, 0.5)
    b = inputs.spinor(L, 95)
    A = bqo.clover_build(U, csw, kappa) if csw else None
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        opts = bq.bq_solve_opts(inner_prec=inner, csw=csw, method=bq.BQ_CGNR)
        info = bq.bq_solve(lat.h, b, x, kappa, 1e-10, opts)
        xb = np.zeros_like(b)
        info_b = bq.bq_solve(lat.h, b, xb, kappa, 1e-10, bq.bq_solve_opts(inner_prec=inner, csw=csw))
    res = oracle_residual(U, x, b, kappa, A=A)
    print(f"cgnr inner={inner} csw={csw}: outer {info.outer_cycles} iters {info.inner_iters} res {res:.2e} (bicgstab iters {info_b.inner_iters})")
    assert info.status == 0 and res <= 1e-10 and abs(res - info.true_rel_residual) < 1e-11
    assert np.linalg.norm(x - xb) / np.linalg.norm(xb) < 1e-8          # both methods reach the same solution
    x_ref, _ = bqo.cgnr(U, b, kappa, tol=1e-12, A=A)
    assert np.linalg.norm(x - x_ref) / np.linalg.norm(x_ref) < 1e-8


def test_cgnr_solve_multi(bq):
    L, kappa, nrhs = (8, 4, 8, 8), 0.1215, 5
    U = inputs.gauge(L, 96, 0.5)
    b = np.stack([inputs.spinor(L, 96 + 100 * k) for k in range(nrhs)])
    b[1] = 0
    x = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        opts = bq.bq_solve_opts(inner_prec=bq.BQ_FP32, method=bq.BQ_CGNR)
        infos = bq.bq_solve_multi(lat.h, b, x, nrhs, kappa, 1e-10, opts)
    for k in range(nrhs):
        assert infos[k].status == 0
        if k == 1:
            assert not x[k].any()
        else:
            assert oracle_residual(U, x[k], b[k], kappa) <= 1e-10
