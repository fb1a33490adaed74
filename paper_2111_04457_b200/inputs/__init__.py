"""Seeded synthetic inputs (gauge links, spinor sources, gauge transforms).

Shared by the oracle's tests and the CUDA path's tests / bench.  Holds none of the method's
arithmetic; see ``gen.c`` for the counter-based recipe.

Canonical layouts, as numpy arrays:
  gauge   U   complex128 [Lt, Lz, Ly, Lx, 4, 3, 3]   (mu = 0..3 = x, y, z, t; U[..., mu, row, col])
  spinor  psi complex128 [Lt, Lz, Ly, Lx, 4, 3]      (spin, colour)
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libbqgen.so")
_STAMP = _LIB + ".stamp"

BASE_SEED = 21110445700  # seed = BASE_SEED + config number (1..5)
STREAM_GAUGE, STREAM_SOURCE, STREAM_TEST, STREAM_GTRANS = 1, 2, 3, 4

_lib = None


def _src_hash() -> str:
    with open(_SRC, "rb") as f:
        return hashlib.sha256(f.read()).hexdigest()


def build(force: bool = False) -> str:
    """Compile gen.c -> libbqgen.so (gcc, OpenMP, no -march so the .so runs on any x86-64 host)."""
    h = _src_hash()
    if not force and os.path.exists(_LIB) and os.path.exists(_STAMP):
        with open(_STAMP) as f:
            if f.read().strip() == h:
                return _LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    with open(_STAMP, "w") as f:
        f.write(h)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        lib.bqgen_su3.argtypes = [ctypes.c_int64, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_double, dp]
        lib.bqgen_su3.restype = None
        lib.bqgen_gauss.argtypes = [ctypes.c_int64, ctypes.c_uint64, ctypes.c_uint64, dp]
        lib.bqgen_gauss.restype = None
        _lib = lib
    return _lib


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def volume(L) -> int:
    Lx, Ly, Lz, Lt = L
    return Lx * Ly * Lz * Lt


def gauge(L, seed: int, eps: float) -> np.ndarray:
    """Links U_mu(x) = reunit(exp(i*eps*H)), H = (G+G^dag)/2 - tr/3, G_ij = N(0,1)+iN(0,1)."""
    Lx, Ly, Lz, Lt = L
    V = volume(L)
    out = np.empty((Lt, Lz, Ly, Lx, 4, 3, 3), dtype=np.complex128)
    _load().bqgen_su3(4 * V, seed, STREAM_GAUGE, float(eps), _dptr(out))
    return out


def unit_gauge(L) -> np.ndarray:
    Lx, Ly, Lz, Lt = L
    out = np.zeros((Lt, Lz, Ly, Lx, 4, 3, 3), dtype=np.complex128)
    out[..., 0, 0] = out[..., 1, 1] = out[..., 2, 2] = 1.0
    return out


def spinor(L, seed: int, stream: int = STREAM_SOURCE) -> np.ndarray:
    """Complex Gaussian source, N(0,1) + i N(0,1) per spin-colour component."""
    Lx, Ly, Lz, Lt = L
    out = np.empty((Lt, Lz, Ly, Lx, 4, 3), dtype=np.complex128)
    _load().bqgen_gauss(12 * volume(L), seed, stream, _dptr(out))
    return out


def gauge_transform(L, seed: int, eps: float = 1.0) -> np.ndarray:
    """One SU(3) matrix g(x) per site, complex128 [Lt, Lz, Ly, Lx, 3, 3]."""
    Lx, Ly, Lz, Lt = L
    out = np.empty((Lt, Lz, Ly, Lx, 3, 3), dtype=np.complex128)
    _load().bqgen_su3(volume(L), seed, STREAM_GTRANS, float(eps), _dptr(out))
    return out


def site_parity(L) -> np.ndarray:
    """(x+y+z+t) & 1 as an int array [Lt, Lz, Ly, Lx] (pure indexing, no arithmetic of the method)."""
    Lx, Ly, Lz, Lt = L
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return (x + y + z + t) & 1
