"""Pins of the oracle's clover term (SURVEY.md §8(c) P3/P4 for clover, P6, P7, P10; readings S4-S6).  CPU only."""
import numpy as np
import pytest

from oracle import bqo
from paper_2111_04457_b200 import inputs
from tests import dense_ref
from tests.conftest import relmax
from tests.test_oracle_pins import gauge_transform_links

T8 = np.diag([1.0, 1.0, -2.0]).astype(complex)


def flux_background(L, k=1):
    """Abelian constant flux in the x-y plane (P6): U_x(x) = exp(-i B y T), U_y = exp(+i B Ly x T) on
    y = Ly-1 else 1, B = 2 pi k/(Lx Ly), T = diag(1,1,-2).  Every x-y plaquette equals exp(i B T)."""
    Lx, Ly, Lz, Lt = L
    B = 2 * np.pi * k / (Lx * Ly)
    U = inputs.unit_gauge(L)
    d = np.diag(T8).real
    for y in range(Ly):
        U[:, :, y, :, 0] = np.diag(np.exp(-1j * B * y * d))
    for x in range(Lx):
        U[:, :, Ly - 1, x, 1] = np.diag(np.exp(1j * B * Ly * x * d))
    return U, B


def test_p6_abelian_flux_field_strength():
    L = (6, 6, 2, 2)
    U, B = flux_background(L)
    F12 = bqo.field_strength(U, 0, 1)
    expect = np.diag([np.sin(B), np.sin(B), -np.sin(2 * B)]).astype(complex)
    assert np.abs(F12 - expect).max() < 1e-15
    assert np.abs(bqo.field_strength(U, 1, 0) + expect).max() < 1e-15   # F_nu_mu = -F_mu_nu
    for mu, nu in ((0, 2), (0, 3), (1, 2), (1, 3), (2, 3)):
        assert np.abs(bqo.field_strength(U, mu, nu)).max() < 1e-15


def test_p7_sign_of_clover_term():
    """At kappa = 1/8 on the flux background the lowest real eigenvalues of D/(2 kappa) sit at ~|qB|/2 for
    csw = 0, return to O(B^2) at csw = +1 (Pauli term cancelled) and double at csw = -1."""
    L = (6, 6, 2, 2)
    kappa = 0.125
    U, B = flux_background(L)
    bc = np.ones(4, dtype=complex)
    low = {}
    for csw in (0.0, 1.0, -1.0):
        A = bqo.clover_build(U, csw, kappa) if csw != 0 else None
        D = dense_ref.dense_dirac(U, kappa, bc=bc, A=A) / (2 * kappa)
        ev = np.linalg.eigvals(D)
        real = np.sort(ev[np.abs(ev.imag) < 1e-9].real)
        low[csw] = real[0]
    assert abs(low[0.0] - B / 2) < 0.1 * B          # ~ |qB|/2 (q = 1 colour components)
    assert abs(low[1.0]) < 0.05 * B                  # O(B^2)
    assert abs(low[-1.0] - B) < 0.1 * B              # doubled


@pytest.fixture(scope="module")
def rough():
    L = (4, 4, 4, 4)
    U = inputs.gauge(L, inputs.BASE_SEED + 4, 0.5)
    return L, U, bqo.clover_build(U, 1.0, 0.1215)


def test_clover_hermitian_trace_gamma5(rough):
    L, U, A = rough
    assert np.abs(A - A.conj().swapaxes(-1, -2)).max() < 1e-15          # PAPER.md:83 "12x12 Hermitian"
    assert np.abs(np.trace(A, axis1=-2, axis2=-1) - 12).max() < 1e-13
    g5 = np.kron(dense_ref.gammas()[4], np.eye(3))
    assert np.abs(A @ g5 - g5 @ A).max() < 1e-15
    assert np.linalg.eigvalsh(A).min() > 0.5                             # positive definite on the configs


def test_clover_csw_kappa_linearity(rough):
    L, U, A = rough
    A2 = bqo.clover_build(U, 2.0, 0.1215)
    assert np.abs((A2 - np.eye(12)) - 2 * (A - np.eye(12))).max() < 1e-14


def test_p4_clover_gauge_covariance(rough):
    L, U, A = rough
    g = inputs.gauge_transform(L, 99)
    Ap = bqo.clover_build(gauge_transform_links(U, g), 1.0, 0.1215)
    G = np.einsum("st,...ab->...satb", np.eye(4), g).reshape(g.shape[:4] + (12, 12))
    assert np.abs(Ap - G @ A @ G.conj().swapaxes(-1, -2)).max() < 1e-13


def test_p3_clover_gamma5_hermiticity_and_dense(rough):
    L, U, A = rough
    kappa = 0.1215
    x = inputs.spinor(L, 5, inputs.STREAM_TEST)
    y = inputs.spinor(L, 5)
    g5 = dense_ref.gammas()[4]
    g5mul = lambda v: np.einsum("st,...tc->...sc", g5, v)
    lhs = np.vdot(x, bqo.dirac_apply(U, y, kappa, A=A))
    rhs = np.vdot(g5mul(bqo.dirac_apply(U, g5mul(x), kappa, A=A)), y)
    assert abs(lhs - rhs) / abs(lhs) < 1e-14
    D = dense_ref.dense_dirac(U, kappa, A=A)
    assert relmax(bqo.dirac_apply(U, y, kappa, A=A), (D @ y.reshape(-1)).reshape(y.shape)) < 1e-14


def test_p10_chirality_blocks(rough):
    """R A R is block diagonal, blocks = 1 + csw kappa sum_k sigma_k (x) (B_k +- E_k)  (Appendix A.4)."""
    L, U, A = rough
    csw, kappa = 1.0, 0.1215
    R = np.kron(np.kron(np.array([[1, 1], [1, -1]]) / np.sqrt(2), np.eye(2)), np.eye(3))
    RAR = R @ A @ R
    assert np.abs(RAR[..., :6, 6:]).max() < 1e-15 and np.abs(RAR[..., 6:, :6]).max() < 1e-15
    F = {(m, n): bqo.field_strength(U, m, n) for m in range(4) for n in range(m + 1, 4)}
    Bf = [F[(1, 2)], -F[(0, 2)], F[(0, 1)]]     # (F23, F31, F12)
    Ef = [F[(0, 3)], F[(1, 3)], F[(2, 3)]]      # (F14, F24, F34)
    sig = [dense_ref.SX, dense_ref.SY, dense_ref.SZ]
    for blk, sgn in ((RAR[..., :6, :6], +1), (RAR[..., 6:, 6:], -1)):
        expect = np.eye(6) + csw * kappa * sum(
            np.einsum("st,...ab->...satb", sig[k], Bf[k] + sgn * Ef[k]).reshape(Bf[k].shape[:4] + (6, 6))
            for k in range(3))
        assert np.abs(blk - expect).max() < 1e-15


def test_site_matrix_invert_and_apply(rough):
    L, U, A = rough
    Ainv = bqo.site_matrix_invert(A)
    assert np.abs(Ainv - np.linalg.inv(A)).max() < 1e-13
    psi = inputs.spinor(L, 6)
    ref = np.einsum("...ij,...j->...i", A, psi.reshape(psi.shape[:4] + (12,))).reshape(psi.shape)
    assert relmax(bqo.site_matrix_apply(A, psi), ref) < 1e-15


def test_p9_clover_schur(rough):
    """Schur complement with clover from masked applies equals the dense block formula; Schur solution
    equals the full dense solve."""
    L, U, A = rough
    kappa = 0.1215
    D = dense_ref.dense_dirac(U, kappa, A=A)
    ie, io = dense_ref.parity_index(L)
    Dee, Deo, Doe, Doo = D[np.ix_(ie, ie)], D[np.ix_(ie, io)], D[np.ix_(io, ie)], D[np.ix_(io, io)]
    M = Dee - Deo @ np.linalg.solve(Doo, Doe)
    b = inputs.spinor(L, 8)
    even = (inputs.site_parity(L) == 0)[..., None, None]
    xe = np.where(even, b, 0)
    got = bqo.schur_apply(U, xe, kappa, A=A, Ainv=bqo.site_matrix_invert(A)).reshape(-1)[ie]
    assert relmax(got, M @ b.reshape(-1)[ie]) < 1e-13
    x, info = bqo.bicgstab(U, b, kappa, tol=1e-12, A=A)
    assert info["status"] == 0
    assert np.linalg.norm(x.reshape(-1) - np.linalg.solve(D, b.reshape(-1))) / np.linalg.norm(x) < 1e-11


# ---------------------------------------------------------------------------------------------------
# P6 in every plane.  test_p6_abelian_flux_field_strength fixes F only in the x-y plane; a mistake in the leaf construction of
# another plane (a transposed pair of directions, a wrong shift, a sign) or in which sigma_mu_nu meets which F_mu_nu would pass
# it.  The same closed form holds in each of the six planes: constant abelian flux B in the (mu, nu) plane.
# ---------------------------------------------------------------------------------------------------
def flux_background_plane(L, mu, nu, k=1):
    """U_mu(x) = exp(-i B x_nu T), U_nu(x) = exp(+i B L_nu x_mu T) on x_nu = L_nu - 1, else 1; B = 2 pi k / (L_mu L_nu), T = diag(1, 1, -2):
    every (mu, nu) plaquette equals exp(i B T), every other plaquette is 1.  Array axes: U[t, z, y, x, direction]."""
    B = 2 * np.pi * k / (L[mu] * L[nu])
    U = inputs.unit_gauge(L)
    d = np.diag(T8).real
    ax = {0: 3, 1: 2, 2: 1, 3: 0}                    # lattice direction -> array axis
    for c in range(L[nu]):
        idx = [slice(None)] * 4
        idx[ax[nu]] = c
        U[tuple(idx) + (mu,)] = np.diag(np.exp(-1j * B * c * d))
    for c in range(L[mu]):
        idx = [slice(None)] * 4
        idx[ax[nu]] = L[nu] - 1
        idx[ax[mu]] = c
        U[tuple(idx) + (nu,)] = np.diag(np.exp(1j * B * L[nu] * c * d))
    return U, B


PLANES = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]


@pytest.mark.parametrize("mu,nu", PLANES)
def test_p6_abelian_flux_in_every_plane(mu, nu):
    L = [2, 2, 2, 2]
    L[mu], L[nu] = 6, 4                               # different extents: a transposed pair of directions changes B
    L = tuple(L)
    U, B = flux_background_plane(L, mu, nu)
    expect = np.diag([np.sin(B), np.sin(B), -np.sin(2 * B)]).astype(complex)
    for a, b in PLANES:
        F = bqo.field_strength(U, a, b)
        if (a, b) == (mu, nu):
            assert np.abs(F - expect).max() < 1e-15, (mu, nu)
            assert np.abs(bqo.field_strength(U, b, a) + expect).max() < 1e-15
        else:
            assert np.abs(F).max() < 1e-15, (mu, nu, a, b)


@pytest.mark.parametrize("mu,nu", PLANES)
def test_clover_matrix_pairs_sigma_with_the_right_plane(mu, nu):
    """On the flux background of plane (mu, nu) the site matrix is exactly 1 - csw kappa sigma_mu_nu (x) diag(sin B, sin B, -sin 2B), with
    sigma_mu_nu = (i/2)[gamma_mu, gamma_nu] built here from the gamma matrices that P1 pins: which sigma multiplies which F, and with
    which sign, in every plane."""
    L = [2, 2, 2, 2]
    L[mu], L[nu] = 6, 4
    L = tuple(L)
    csw, kappa = 1.3, 0.11
    U, B = flux_background_plane(L, mu, nu)
    g = [bqo.gamma(m) for m in range(4)]
    sig = 0.5j * (g[mu] @ g[nu] - g[nu] @ g[mu])
    F = np.diag([np.sin(B), np.sin(B), -np.sin(2 * B)]).astype(complex)
    expect = np.eye(12) - csw * kappa * np.kron(sig, F)          # index = 3 * spin + colour
    A = bqo.clover_build(U, csw, kappa)
    assert np.abs(A - expect).max() < 1e-14, (mu, nu)


def test_traceless_option_removes_exactly_the_trace():
    """Reading S5 keeps the trace of F_mu_nu (the default everywhere in this repository).  The oracle's optional `traceless`
    branch is pinned to the pinned default: F' = F - (tr F / 3) 1 in every plane on every site, tr F' = 0, and — since
    sigma_mu_nu is traceless — the site trace of the clover matrix A is 12 either way, while A itself differs where tr F != 0.
    An abelian U(1)^3 field (phases not summing to zero per link) has tr F != 0, so the branch is exercised, not vacuous."""
    L = (4, 4, 2, 2)
    rng = np.random.default_rng(77)
    Lx, Ly, Lz, Lt = L
    ph = rng.uniform(-0.6, 0.6, size=(Lt, Lz, Ly, Lx, 4, 3))
    U = np.zeros((Lt, Lz, Ly, Lx, 4, 3, 3), dtype=np.complex128)
    for c in range(3):
        U[..., c, c] = np.exp(1j * ph[..., c])
    eye = np.eye(3)
    saw_trace = False
    for mu in range(4):
        for nu in range(mu + 1, 4):
            F = bqo.field_strength(U, mu, nu)
            Ft = bqo.field_strength(U, mu, nu, traceless=True)
            tr = np.trace(F, axis1=-2, axis2=-1)
            saw_trace = saw_trace or np.abs(tr).max() > 1e-3
            assert np.abs(Ft - (F - tr[..., None, None] / 3.0 * eye)).max() < 1e-14
            assert np.abs(np.trace(Ft, axis1=-2, axis2=-1)).max() < 1e-14
    assert saw_trace
    A, At = bqo.clover_build(U, 1.3, 0.12), bqo.clover_build(U, 1.3, 0.12, traceless=True)
    assert np.abs(np.trace(A, axis1=-2, axis2=-1) - 12).max() < 1e-12 and np.abs(np.trace(At, axis1=-2, axis2=-1) - 12).max() < 1e-12
    assert np.abs(A - At).max() > 1e-4
