"""oracle/bqo.py — TEST INFRASTRUCTURE, NOT PRODUCT.

numpy-facing wrapper of ``bqo.c``: the plain double-precision CPU Dirac operator (Eq. 1,
PAPER.md:81) and textbook BiCGStab.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It imports nothing from the CUDA package.

Array conventions:
  L = (Lx, Ly, Lz, Lt); U complex128 [Lt,Lz,Ly,Lx,4,3,3]; psi complex128 [Lt,Lz,Ly,Lx,4,3];
  site-diagonal matrices A complex128 [Lt,Lz,Ly,Lx,12,12] (index 3*spin+colour);
  bc = 4 complex boundary phases (default periodic x,y,z, antiperiodic t: BASELINE.json config 1).

The even-odd quantities (reading O3) are built here from MASKED FULL-LATTICE applies — the oracle
has no checkerboard code: (-kappa H_eo psi_o) = (D [0; psi_o])_e.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bqo.c")
_LIB = os.path.join(_HERE, "libbqo.so")
_STAMP = _LIB + ".stamp"

DEFAULT_BC = (1.0 + 0j, 1.0 + 0j, 1.0 + 0j, -1.0 + 0j)

_lib = None
_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)
_lp = ctypes.POINTER(ctypes.c_long)


def build(force: bool = False) -> str:
    """gcc -O3 -fopenmp, no -march (the .so must run on whatever x86-64 host the GPU box has)."""
    with open(_SRC, "rb") as f:
        h = hashlib.sha256(f.read()).hexdigest()
    if not force and os.path.exists(_LIB) and os.path.exists(_STAMP):
        with open(_STAMP) as f:
            if f.read().strip() == h:
                return _LIB
    cmd = ["gcc", "-O3", "-std=c99", "-fopenmp", "-fcx-limited-range", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    with open(_STAMP, "w") as f:
        f.write(h)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.bqo_gamma.argtypes = [ctypes.c_int, _dp]
        lib.bqo_gamma.restype = None
        lib.bqo_dirac_apply.argtypes = [_ip, _dp, _dp, ctypes.c_double, _dp, _dp, _dp]
        lib.bqo_dirac_apply_dag.argtypes = [_ip, _dp, _dp, ctypes.c_double, _dp, _dp, _dp]
        lib.bqo_dirac_apply_sites.argtypes = [_ip, _dp, _dp, ctypes.c_double, _dp, _dp, ctypes.c_long, _lp, _dp]
        lib.bqo_field_strength.argtypes = [_ip, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp]
        lib.bqo_clover_build.argtypes = [_ip, _dp, ctypes.c_double, ctypes.c_double, ctypes.c_int, _dp]
        lib.bqo_site_matrix_invert.argtypes = [ctypes.c_long, _dp, _dp]
        lib.bqo_site_matrix_apply.argtypes = [ctypes.c_long, _dp, _dp, _dp]
        lib.bqo_bicgstab.argtypes = [_ip, _dp, _dp, ctypes.c_double, _dp, _dp, _dp, ctypes.c_double, ctypes.c_int,
                                     _ip, _dp, _ip]
        lib.bqo_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


def _Larr(L):
    return (ctypes.c_int * 4)(*[int(v) for v in L])


def _bc(bc):
    return _c(np.asarray(DEFAULT_BC if bc is None else bc, dtype=np.complex128))


def lattice_of(psi_or_U):
    Lt, Lz, Ly, Lx = psi_or_U.shape[:4]
    return (Lx, Ly, Lz, Lt)


def num_threads() -> int:
    return int(_load().bqo_num_threads())


def gamma(mu: int) -> np.ndarray:
    """gamma_mu (mu = 0..3 = x,y,z,t) or gamma_5 (mu = 4) as a 4x4 complex matrix."""
    out = np.empty((4, 4), dtype=np.complex128)
    _load().bqo_gamma(mu, _p(out))
    return out


def dirac_apply(U, psi, kappa, bc=None, A=None) -> np.ndarray:
    """out = D psi (Eq. 1).  A = None: Wilson (F = 0); else the dense site-diagonal term 1 + F(x)."""
    U, psi = _c(U), _c(psi)
    L = lattice_of(psi)
    out = np.empty_like(psi)
    bcv = _bc(bc)
    Ac = None if A is None else _c(A)
    _load().bqo_dirac_apply(_Larr(L), _p(bcv), _p(U), float(kappa), _p(Ac), _p(psi), _p(out))
    return out


def dirac_apply_dag(U, psi, kappa, bc=None, A=None) -> np.ndarray:
    """out = D^dagger psi, by the definition of the adjoint (scatter of the conjugate-transposed blocks of Eq. 1)."""
    U, psi = _c(U), _c(psi)
    L = lattice_of(psi)
    out = np.empty_like(psi)
    bcv = _bc(bc)
    Ac = None if A is None else _c(A)
    _load().bqo_dirac_apply_dag(_Larr(L), _p(bcv), _p(U), float(kappa), _p(Ac), _p(psi), _p(out))
    return out


def cgnr(U, b, kappa, tol=1e-12, max_iter=10000, bc=None, A=None):
    """Solve D x = b by conjugate gradients on the normal equations D^dag D x = D^dag b (Hestenes-Stiefel CG,
    textbook form).  Stops when the TRUE residual of the original system satisfies
    |b - D x| / |b| <= tol (checked every iteration with its own operator apply: slow and obviously right).
    Returns (x, info dict)."""
    b = _c(b)
    x = np.zeros_like(b)
    bnorm = np.linalg.norm(b)
    if bnorm == 0.0:
        return x, {"status": 0, "iters": 0, "relres": 0.0}
    r = dirac_apply_dag(U, b, kappa, bc=bc, A=A)        # normal-equation residual D^dag (b - D x), x = 0
    p = r.copy()
    rr = np.vdot(r, r).real
    status, it, rel = 1, 0, 1.0
    while it < max_iter:
        q = dirac_apply(U, p, kappa, bc=bc, A=A)
        alpha = rr / np.vdot(q, q).real                 # <p, D^dag D p> = |D p|^2
        x = x + alpha * p
        r = r - alpha * dirac_apply_dag(U, q, kappa, bc=bc, A=A)
        it += 1
        rel = np.linalg.norm(b - dirac_apply(U, x, kappa, bc=bc, A=A)) / bnorm
        if rel <= tol:
            status = 0
            break
        rr_new = np.vdot(r, r).real
        p = r + (rr_new / rr) * p
        rr = rr_new
    return x, {"status": status, "iters": it, "relres": rel}


def dirac_apply_sites(U, psi, kappa, sites, bc=None, A=None) -> np.ndarray:
    """(D psi)(x) at the canonical site indices `sites` only -> [nsites, 4, 3]."""
    U, psi = _c(U), _c(psi)
    L = lattice_of(psi)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((len(sites), 4, 3), dtype=np.complex128)
    bcv = _bc(bc)
    Ac = None if A is None else _c(A)
    _load().bqo_dirac_apply_sites(_Larr(L), _p(bcv), _p(U), float(kappa), _p(Ac), _p(psi), len(sites),
                                  sites.ctypes.data_as(_lp), _p(out))
    return out


def field_strength(U, mu, nu, traceless=False) -> np.ndarray:
    """F_mu_nu(x) = (Q - Q^dag)/(8i), Q = four leaves (Appendix A.3) -> [Lt,Lz,Ly,Lx,3,3]."""
    U = _c(U)
    L = lattice_of(U)
    out = np.empty(U.shape[:4] + (3, 3), dtype=np.complex128)
    _load().bqo_field_strength(_Larr(L), _p(U), mu, nu, int(traceless), _p(out))
    return out


def clover_build(U, csw, kappa, traceless=False) -> np.ndarray:
    """A(x) = 1 - csw*kappa*sum_{mu<nu} sigma_mu_nu (x) F_mu_nu(x), dense [Lt,Lz,Ly,Lx,12,12]."""
    U = _c(U)
    L = lattice_of(U)
    out = np.empty(U.shape[:4] + (12, 12), dtype=np.complex128)
    _load().bqo_clover_build(_Larr(L), _p(U), float(csw), float(kappa), int(traceless), _p(out))
    return out


def site_matrix_invert(A) -> np.ndarray:
    A = _c(A)
    V = int(np.prod(A.shape[:-2]))
    out = np.empty_like(A)
    nsing = _load().bqo_site_matrix_invert(V, _p(A), _p(out))
    if nsing:
        raise np.linalg.LinAlgError(f"{nsing} singular site matrices")
    return out


def site_matrix_apply(A, psi) -> np.ndarray:
    A, psi = _c(A), _c(psi)
    V = int(np.prod(A.shape[:-2]))
    out = np.empty_like(psi)
    _load().bqo_site_matrix_apply(V, _p(A), _p(psi), _p(out))
    return out


def bicgstab(U, b, kappa, tol=1e-12, max_iter=10000, bc=None, A=None, x0=None):
    """Solve D x = b on the full lattice (reading O4).  Returns (x, info dict)."""
    U, b = _c(U), _c(b)
    L = lattice_of(b)
    x = np.zeros_like(b) if x0 is None else _c(x0).copy()
    bcv = _bc(bc)
    Ac = None if A is None else _c(A)
    iters = ctypes.c_int(0)
    restarts = ctypes.c_int(0)
    relres = ctypes.c_double(0)
    status = _load().bqo_bicgstab(_Larr(L), _p(bcv), _p(U), float(kappa), _p(Ac), _p(b), _p(x), float(tol),
                                  int(max_iter), ctypes.byref(iters), ctypes.byref(relres), ctypes.byref(restarts))
    return x, {"status": int(status), "iters": iters.value, "relres": relres.value, "restarts": restarts.value}


# ---- even-odd quantities from masked full-lattice applies (reading O3) ------------------------------

def parity_mask(L) -> np.ndarray:
    Lx, Ly, Lz, Lt = L
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return (x + y + z + t) & 1


def hop_restricted(U, psi, kappa, out_parity, bc=None) -> np.ndarray:
    """-kappa H_{p,1-p} psi_{1-p} as a full-lattice array that is zero on parity 1-p sites:
    (D [psi restricted to parity 1-p])_p  (Wilson D has D_pp = 1, so the diagonal does not contribute)."""
    L = lattice_of(psi)
    par = parity_mask(L)
    masked = np.where((par == (1 - out_parity))[..., None, None], psi, 0)
    full = dirac_apply(U, masked, kappa, bc=bc)
    return np.where((par == out_parity)[..., None, None], full, 0)


def schur_apply(U, psi_e, kappa, bc=None, A=None, Ainv=None) -> np.ndarray:
    """M^ x_e = A_ee x_e - kappa^2 H_eo A_oo^-1 H_oe x_e on a full-lattice array supported on EVEN sites."""
    L = lattice_of(psi_e)
    par = parity_mask(L)
    even = (par == 0)[..., None, None]
    xe = np.where(even, psi_e, 0)
    y = dirac_apply(U, xe, kappa, bc=bc, A=A)          # even: A_ee x_e ; odd: -kappa H_oe x_e
    y_e = np.where(even, y, 0)
    y_o = np.where(~even, y, 0)
    if Ainv is not None:
        y_o = site_matrix_apply(Ainv, y_o)
    z = dirac_apply(U, y_o, kappa, bc=bc, A=A)          # even part: -kappa H_eo (A_oo^-1)(-kappa H_oe x_e)
    return y_e - np.where(even, z, 0)
