"""Brute-force dense Wilson(-clover) matrix in numpy — a code path disjoint from oracle/bqo.c.

Used only by the `-m "not gpu"` pins.  The gamma matrices are built here
from Pauli matrices with Kronecker products (Appendix A.1: gamma_k = [[0,-i s_k],[+i s_k,0]] =
sigma_y (x) sigma_k, gamma_4 = sigma_z (x) 1), NOT copied from the oracle's 4x4 tables; the hopping
term is assembled by fancy-index assignment of kron((1 -+ gamma_mu), U) blocks into a
[V,4,3,V,4,3] tensor, with neighbour tables from np.roll of an index grid.
"""
import numpy as np

S0 = np.eye(2, dtype=complex)
SX = np.array([[0, 1], [1, 0]], dtype=complex)
SY = np.array([[0, -1j], [1j, 0]], dtype=complex)
SZ = np.array([[1, 0], [0, -1]], dtype=complex)


def gammas():
    """[gx, gy, gz, gt, g5]; sigma_y (x) sigma_k = [[0, -i s_k], [i s_k, 0]]."""
    g = [np.kron(SY, s) for s in (SX, SY, SZ)] + [np.kron(SZ, S0)]
    g5 = g[0] @ g[1] @ g[2] @ g[3]
    return g + [g5]


def neighbour_tables(L, bc):
    """fwd[mu][s], bwd[mu][s] (canonical site indices) and the phases phi+[mu][s], phi-[mu][s]."""
    Lx, Ly, Lz, Lt = L
    V = Lx * Ly * Lz * Lt
    grid = np.arange(V).reshape(Lt, Lz, Ly, Lx)
    coords = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    fwd, bwd, pf, pb = [], [], [], []
    for mu in range(4):
        ax = 3 - mu
        fwd.append(np.roll(grid, -1, axis=ax).ravel())
        bwd.append(np.roll(grid, +1, axis=ax).ravel())
        c = coords[ax].ravel()
        pf.append(np.where(c == L[mu] - 1, bc[mu], 1.0 + 0j))
        pb.append(np.where(c == 0, np.conj(bc[mu]), 1.0 + 0j))
    return fwd, bwd, pf, pb


def dense_dirac(U, kappa, bc=(1, 1, 1, -1), A=None):
    """D as a (12V x 12V) complex matrix, row/col index = 12*s + 3*spin + colour."""
    Lt, Lz, Ly, Lx = U.shape[:4]
    L = (Lx, Ly, Lz, Lt)
    V = Lx * Ly * Lz * Lt
    bc = np.asarray(bc, dtype=complex)
    g = gammas()
    Us = U.reshape(V, 4, 3, 3)
    fwd, bwd, pf, pb = neighbour_tables(L, bc)
    D = np.zeros((V, 4, 3, V, 4, 3), dtype=complex)
    idx = np.arange(V)
    if A is None:
        D[idx, :, :, idx, :, :] += np.einsum("st,ab->satb", np.eye(4), np.eye(3))[None]
    else:
        D[idx, :, :, idx, :, :] += A.reshape(V, 4, 3, 4, 3)
    one = np.eye(4)
    for mu in range(4):
        Uf = Us[:, mu]                                   # U_mu(x)
        Ub = Us[bwd[mu], mu].conj().transpose(0, 2, 1)   # U_mu(x - mu)^dagger
        D[idx, :, :, fwd[mu], :, :] += -kappa * pf[mu][:, None, None, None, None] * np.einsum(
            "st,xab->xsatb", one - g[mu], Uf)
        D[idx, :, :, bwd[mu], :, :] += -kappa * pb[mu][:, None, None, None, None] * np.einsum(
            "st,xab->xsatb", one + g[mu], Ub)
    return D.reshape(12 * V, 12 * V)


def parity_index(L):
    """Dense row indices (12 per site) of the even and odd sites."""
    Lx, Ly, Lz, Lt = L
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    par = ((x + y + z + t) & 1).ravel()
    rows = np.arange(12 * par.size).reshape(-1, 12)
    return rows[par == 0].ravel(), rows[par == 1].ravel()
