"""Pins of the oracle's D^dagger and CGNR (PAPER.md:44 set_mode) against what theory fixes:
the conjugate transpose of the brute-force dense matrix (tests/dense_ref.py, a code path disjoint from oracle/bqo.c),
gamma5-hermiticity D^dag = g5 D g5, the free-field closed form (eigenvalue conj(lambda)), the point-source stencil,
and numpy.linalg.solve for the normal-equation solver.  CPU only."""
import numpy as np
import pytest

from oracle import bqo
from paper_2111_04457_b200 import inputs
from tests import dense_ref
from tests.conftest import relmax

BC = np.array([1, 1, 1, -1], dtype=complex)
GENERAL_BC = np.exp(1j * np.array([0.4, -1.3, 2.0, 0.9]))


@pytest.fixture(scope="module")
def dense44(cfg1):
    return dense_ref.dense_dirac(cfg1["U"], cfg1["kappa"], bc=BC)


def test_dagger_is_conjugate_transpose_of_dense(cfg1, dense44):
    psi = cfg1["b"]
    ref = (dense44.conj().T @ psi.reshape(-1)).reshape(psi.shape)
    assert relmax(bqo.dirac_apply_dag(cfg1["U"], psi, cfg1["kappa"]), ref) < 1e-14


def test_dagger_dense_general_phases_and_clover():
    """Complex phases in every direction, an L = 2 direction, and a (Hermitian) clover term."""
    L = (4, 2, 6, 2)
    U = inputs.gauge(L, 78, 0.6)
    psi = inputs.spinor(L, 78)
    A = bqo.clover_build(U, 1.0, 0.13)
    for Aterm in (None, A):
        D = dense_ref.dense_dirac(U, 0.13, bc=GENERAL_BC, A=Aterm)
        ref = (D.conj().T @ psi.reshape(-1)).reshape(psi.shape)
        assert relmax(bqo.dirac_apply_dag(U, psi, 0.13, bc=GENERAL_BC, A=Aterm), ref) < 1e-14


@pytest.mark.parametrize("bc", [None, GENERAL_BC])
def test_dagger_gamma5_hermiticity(bc):
    """D^dag = g5 D g5 (the identity the CUDA kernel's dagger mode is built on), Wilson and clover."""
    L = (4, 4, 2, 6)
    U = inputs.gauge(L, 79, 0.5)
    psi = inputs.spinor(L, 79)
    g5 = dense_ref.gammas()[4]
    g5mul = lambda v: np.einsum("st,...tc->...sc", g5, v)
    for A in (None, bqo.clover_build(U, 1.0, 0.12)):
        lhs = bqo.dirac_apply_dag(U, psi, 0.12, bc=bc, A=A)
        rhs = g5mul(bqo.dirac_apply(U, g5mul(psi), 0.12, bc=bc, A=A))
        assert relmax(lhs, rhs) < 1e-14


def test_dagger_adjointness_random_vectors():
    L = (6, 4, 4, 2)
    U = inputs.gauge(L, 80, 0.7)
    x, y = inputs.spinor(L, 80), inputs.spinor(L, 81, inputs.STREAM_TEST)
    lhs = np.vdot(x, bqo.dirac_apply(U, y, 0.124, bc=GENERAL_BC))
    rhs = np.vdot(bqo.dirac_apply_dag(U, x, 0.124, bc=GENERAL_BC), y)
    assert abs(lhs - rhs) / abs(lhs) < 1e-14


def test_dagger_free_field_plane_wave():
    """U = 1: D psi = lambda psi for a plane-wave eigen-spinor; D is normal there, so D^dag psi = conj(lambda) psi,
    lambda = 1 - 2 kappa sum cos p +- 2 i kappa sqrt(sum sin^2 p)."""
    L, kappa = (4, 6, 4, 8), 0.11
    Lx, Ly, Lz, Lt = L
    U = np.zeros((Lt, Lz, Ly, Lx, 4, 3, 3), dtype=complex)
    U[..., np.arange(3), np.arange(3)] = 1
    theta = np.array([0, 0, 0, np.pi])                      # antiperiodic in t
    n = np.array([1, 2, 3, 5])
    p = (2 * np.pi * n + theta) / np.array(L)
    g = dense_ref.gammas()
    M = 1j * sum(g[mu] * np.sin(p[mu]) for mu in range(4))   # i sum gamma_mu sin p_mu, anti-Hermitian
    ev, vec = np.linalg.eig(M)
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    wave = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    for k in range(4):
        u = np.einsum("s,c->sc", vec[:, k], np.array([1.0, -0.5j, 0.25]))
        psi = wave[..., None, None] * u
        lam = 1 - 2 * kappa * np.cos(p).sum() + 2 * kappa * ev[k]
        assert relmax(bqo.dirac_apply(U, psi, kappa), lam * psi) < 1e-13
        assert relmax(bqo.dirac_apply_dag(U, psi, kappa), np.conj(lam) * psi) < 1e-13
        assert abs(abs(ev[k]) - np.sqrt((np.sin(p) ** 2).sum())) < 1e-13


def test_dagger_point_source():
    """delta source e_s (x) e_c at the origin on U = 1: D^dag puts -kappa phi (1+g_mu)[:,s] on the site -mu^ (whose forward
    neighbour is the origin) — the projectors of D exchanged; with s = 0 and mu = t, (1+g_4) keeps the upper spins:
    site -t^ gets -2 kappa * (-1) (antiperiodic wrap), site +t^ gets 0."""
    L, kappa = (4, 4, 4, 4), 0.12
    U = np.zeros((4, 4, 4, 4, 4, 3, 3), dtype=complex)
    U[..., np.arange(3), np.arange(3)] = 1
    psi = np.zeros((4, 4, 4, 4, 4, 3), dtype=complex)
    psi[0, 0, 0, 0, 0, 1] = 1
    out = bqo.dirac_apply_dag(U, psi, kappa)
    assert out[0, 0, 0, 0, 0, 1] == 1
    assert abs(out[3, 0, 0, 0, 0, 1] - 2 * kappa) < 1e-15 and np.abs(out[1, 0, 0, 0]).max() == 0
    g = dense_ref.gammas()
    assert np.allclose(out[0, 0, 0, 3, :, 1], -kappa * (np.eye(4) + g[0])[:, 0])     # site -x^
    assert np.allclose(out[0, 0, 0, 1, :, 1], -kappa * (np.eye(4) - g[0])[:, 0])     # site +x^


def test_cgnr_vs_linalg_solve(cfg1, dense44):
    b = cfg1["b"]
    x_ref = np.linalg.solve(dense44, b.reshape(-1)).reshape(b.shape)
    x, info = bqo.cgnr(cfg1["U"], b, cfg1["kappa"], tol=1e-12)
    assert info["status"] == 0 and info["relres"] <= 1e-12
    assert np.linalg.norm(x - x_ref) / np.linalg.norm(x_ref) < 1e-11
    assert np.linalg.norm(b.reshape(-1) - dense44 @ x.reshape(-1)) / np.linalg.norm(b) < 2e-12
