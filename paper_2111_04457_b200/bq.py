"""Thin ctypes binding of libbq.so (include/bq.h; test and benchmark hooks: include/bq_test.h) — argument marshalling only.

Every function has the name and argument order of its C counterpart; every step of the path runs in the
library's CUDA kernels.  torch is used only to own device memory (tensors -> raw pointers) and streams.
There is no CPU fallback: importing works without a GPU (so that symbol checks can run), but every compute
call raises BqError (BQ_ECUDA) when no device is present, and loading fails loudly if libbq.so is missing.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("BQ_LIB", os.path.join(_HERE, "libbq.so"))   # BQ_LIB: load another build of the same library

# enums (include/bq.h)
BQ_OK, BQ_EINVAL, BQ_EODD_EXTENT, BQ_ENOGAUGE, BQ_ENOCLOVER, BQ_ESINGULAR_CLOVER, BQ_ECUDA, BQ_ENOMEM, \
    BQ_ENOTCONVERGED, BQ_EBREAKDOWN = range(10)
BQ_FP64, BQ_FP32, BQ_HALF = 0, 1, 2
BQ_EVEN, BQ_ODD, BQ_FULL = 0, 1, 2
BQ_RECON18, BQ_RECON12 = 0, 1
BQ_MODE_D, BQ_MODE_DDAG, BQ_MODE_DDAGD = 0, 1, 2
BQ_BICGSTAB, BQ_CGNR = 0, 1

EXPORTS = [
    "bq_lattice_create", "bq_lattice_destroy", "bq_status_string", "bq_last_error", "bq_gauge_load",
    "bq_field_bytes", "bq_field_import", "bq_field_export", "bq_wilson_apply", "bq_clover_apply",
    "bq_dirac_apply", "bq_schur_apply", "bq_solve", "bq_blas_norm2", "bq_blas_cdot", "bq_blas_caxpy",
    "bq_blas_bicg_update", "bq_get_counters", "bq_bench_kernel", "bq_schur_apply_dots",
    "bq_wilson_apply_multi", "bq_schur_apply_multi", "bq_bench_kernel_multi", "bq_solve_multi", "bq_dirac_apply_mode", "bq_schur_apply_mode", "bq_propagator",
    "bq_lattice_create_sub", "bq_dd_face_bytes", "bq_dd_pack", "bq_dd_unpack", "bq_dd_wilson_apply", "bq_dd_solve",
    "bq_field_norm2_noalloc",
]


class bq_solve_opts(ctypes.Structure):
    _fields_ = [("inner_prec", ctypes.c_int), ("recon", ctypes.c_int), ("csw", ctypes.c_double),
                ("inner_tol", ctypes.c_double), ("max_inner", ctypes.c_int), ("max_outer", ctypes.c_int),
                ("check_every", ctypes.c_int), ("method", ctypes.c_int), ("lexical", ctypes.c_int), ("x0_zero", ctypes.c_int), ("stream", ctypes.c_void_p)]


class bq_solve_info(ctypes.Structure):
    _fields_ = [("status", ctypes.c_int), ("outer_cycles", ctypes.c_int), ("inner_iters", ctypes.c_int),
                ("restarts", ctypes.c_int), ("true_rel_residual", ctypes.c_double), ("seconds", ctypes.c_double),
                ("phase_seconds", ctypes.c_double * 5)]


class BqError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"bq status {status}: {msg}")
        self.status = status


_lib = None
_vp, _dp, _i, _d = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_double


def lib():
    """Load libbq.so (build it first with `python -m paper_2111_04457_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: run `python -m paper_2111_04457_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        L.bq_lattice_create.argtypes = [_i, _i, _i, _i, _dp, ctypes.POINTER(_vp)]
        L.bq_lattice_destroy.argtypes = [_vp]
        L.bq_status_string.argtypes = [_i]
        L.bq_status_string.restype = ctypes.c_char_p
        L.bq_last_error.argtypes = [_vp]
        L.bq_last_error.restype = ctypes.c_char_p
        L.bq_gauge_load.argtypes = [_vp, _vp]
        L.bq_field_bytes.argtypes = [_vp, _i, _i, ctypes.POINTER(ctypes.c_size_t)]
        L.bq_field_import.argtypes = [_vp, _vp, _vp, _i, _i, _vp]
        L.bq_field_export.argtypes = [_vp, _vp, _vp, _i, _i, _vp]
        L.bq_wilson_apply.argtypes = [_vp, _vp, _vp, _d, _i, _i, _i, _vp]
        L.bq_clover_apply.argtypes = [_vp, _d, _d, _vp, _vp, _i, _i, _i, _vp]
        L.bq_dirac_apply.argtypes = [_vp, _vp, _vp, _d, _d, _i, _i, _vp]
        L.bq_schur_apply.argtypes = [_vp, _vp, _vp, _vp, _d, _d, _i, _i, _vp]
        L.bq_schur_apply_dots.argtypes = [_vp, _vp, _vp, _vp, _d, _d, _i, _i, _vp, _dp]
        L.bq_solve.argtypes = [_vp, _vp, _vp, _d, _d, ctypes.POINTER(bq_solve_opts), ctypes.POINTER(bq_solve_info)]
        L.bq_solve_multi.argtypes = [_vp, _vp, _vp, _i, _d, _d, ctypes.POINTER(bq_solve_opts), ctypes.POINTER(bq_solve_info)]
        L.bq_propagator.argtypes = [_vp, ctypes.POINTER(_i), _vp, _d, _d, ctypes.POINTER(bq_solve_opts), ctypes.POINTER(bq_solve_info)]
        L.bq_dirac_apply_mode.argtypes = [_vp, _vp, _vp, _vp, _d, _d, _i, _i, _i, _vp]
        L.bq_schur_apply_mode.argtypes = [_vp, _vp, _vp, _vp, _vp, _d, _d, _i, _i, _i, _vp]
        L.bq_blas_norm2.argtypes = [_vp, _vp, _i, _dp]
        L.bq_blas_cdot.argtypes = [_vp, _vp, _vp, _i, _dp]
        L.bq_blas_caxpy.argtypes = [_vp, _dp, _vp, _vp, _i]
        L.bq_blas_bicg_update.argtypes = [_vp, _dp, _dp, _vp, _vp, _vp, _vp, _vp, _vp, _i, _dp, _dp]
        L.bq_get_counters.argtypes = [_vp, ctypes.POINTER(ctypes.c_ulonglong)]
        L.bq_bench_kernel.argtypes = [_vp, _i, _i, _i, _d, _d, _i, _i, _dp, _dp]
        L.bq_wilson_apply_multi.argtypes = [_vp, _vp, _vp, _i, _d, _i, _i, _i, _vp]
        L.bq_schur_apply_multi.argtypes = [_vp, _vp, _vp, _vp, _i, _d, _d, _i, _i, _vp]
        L.bq_bench_kernel_multi.argtypes = [_vp, _i, _i, _i, _d, _d, _i, _i, _i, _dp, _dp]
        _pp = ctypes.POINTER(_vp)
        L.bq_lattice_create_sub.argtypes = [_i, _i, _i, _i, _dp, ctypes.POINTER(_i), ctypes.POINTER(_i), ctypes.POINTER(_vp)]
        L.bq_dd_face_bytes.argtypes = [_vp, _i, _i, ctypes.POINTER(ctypes.c_size_t)]
        L.bq_dd_pack.argtypes = [_vp, _pp, _vp, _i, _i, _i, _vp]
        L.bq_dd_unpack.argtypes = [_vp, _vp, _pp, _d, _i, _i, _i, _vp]
        L.bq_dd_wilson_apply.argtypes = [_pp, _i, _pp, _pp, _d, _i, _i, _i, _vp]
        L.bq_dd_solve.argtypes = [_pp, _i, _pp, _pp, _d, _d, _i, ctypes.POINTER(bq_solve_info)]
        L.bq_field_norm2_noalloc.argtypes = [_vp, ctypes.c_longlong, _i, _vp, _vp, ctypes.c_char_p, ctypes.c_size_t]
        for name in EXPORTS:
            if name not in ("bq_status_string", "bq_last_error"):
                getattr(L, name).restype = _i
        _lib = L
    return _lib


def _ptr(t):
    """Raw pointer of a torch tensor / numpy array / int / None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


_DIMS = {}       # handle -> (Lx, Ly, Lz, Lt), recorded by bq_lattice_create: sizes the canonical arrays are checked against


def _canonical(h, a, nfields, name, reals_per_site=24):
    """Pointer of a canonical fp64 array after checking what the C side cannot: dtype complex128 / float64, C-contiguous,
    nfields * reals_per_site * V doubles.  Nothing is copied or converted: a wrong array is an error (BQ_EINVAL), not a guess."""
    if isinstance(a, int) or a is None:
        return a
    if isinstance(a, np.ndarray):
        per = {np.dtype(np.complex128): 2.0, np.dtype(np.float64): 1.0, np.dtype(np.uint8): 0.125}.get(a.dtype)
        contiguous, n = a.flags["C_CONTIGUOUS"], a.size
    else:
        import torch
        per = {torch.complex128: 2.0, torch.float64: 1.0, torch.uint8: 0.125}.get(a.dtype)
        contiguous, n = a.is_contiguous(), a.numel()
    if per is None:
        raise BqError(BQ_EINVAL, f"{name}: dtype must be complex128 (or float64, or raw uint8 bytes), got {a.dtype}")
    doubles = n * per
    if not contiguous:
        raise BqError(BQ_EINVAL, f"{name}: array must be C-contiguous")
    dims = _DIMS.get(h.value if hasattr(h, "value") else h)
    if dims is not None:
        want = nfields * reals_per_site * dims[0] * dims[1] * dims[2] * dims[3]
        if doubles != want:
            raise BqError(BQ_EINVAL, f"{name}: {doubles} doubles, expected {want} ({nfields} field(s) of {reals_per_site} reals x V)")
    return _ptr(a)


def _check(h, st, allow=()):
    if st != BQ_OK and st not in allow:
        msg = lib().bq_last_error(h).decode() if h else ""
        raise BqError(st, f"{lib().bq_status_string(st).decode()}: {msg}")
    return st


def _stream_ptr(stream):
    if stream is None:
        return None
    return stream if isinstance(stream, int) else stream.cuda_stream


# ---- the C calls, same names ----------------------------------------------------------------------
def bq_lattice_create(Lx, Ly, Lz, Lt, bc_phase=None):
    h = _vp()
    bc = None
    if bc_phase is not None:
        arr = np.asarray(bc_phase, dtype=np.complex128).view(np.float64)
        bc = (ctypes.c_double * 8)(*arr)
    st = lib().bq_lattice_create(Lx, Ly, Lz, Lt, bc, ctypes.byref(h))
    if st != BQ_OK:
        raise BqError(st, lib().bq_status_string(st).decode())
    _DIMS[h.value] = (int(Lx), int(Ly), int(Lz), int(Lt))
    return h


def bq_lattice_destroy(h):
    _DIMS.pop(h.value if hasattr(h, "value") else h, None)
    return lib().bq_lattice_destroy(h)


def bq_gauge_load(h, U):
    """U: canonical complex128 [Lt,Lz,Ly,Lx,4,3,3] numpy array (host) or torch CUDA tensor."""
    if isinstance(U, np.ndarray):
        U = np.ascontiguousarray(U, dtype=np.complex128)
    _check(h, lib().bq_gauge_load(h, _ptr(U)))


def bq_field_bytes(h, prec, parity):
    n = ctypes.c_size_t(0)
    _check(h, lib().bq_field_bytes(h, prec, parity, ctypes.byref(n)))
    return n.value


def bq_field_import(h, internal, canonical, parity, prec, stream=None):
    _check(h, lib().bq_field_import(h, _ptr(internal), _canonical(h, canonical, 1, "canonical"), parity, prec, _stream_ptr(stream)))


def bq_field_export(h, canonical, internal, parity, prec, stream=None):
    _check(h, lib().bq_field_export(h, _canonical(h, canonical, 1, "canonical"), _ptr(internal), parity, prec, _stream_ptr(stream)))


def bq_wilson_apply(h, out, inp, kappa, parity, prec=BQ_FP32, recon=BQ_RECON18, stream=None):
    _check(h, lib().bq_wilson_apply(h, _ptr(out), _ptr(inp), kappa, parity, prec, recon, _stream_ptr(stream)))


def bq_clover_apply(h, csw, kappa, out, inp, parity, inverse, prec, stream=None):
    _check(h, lib().bq_clover_apply(h, csw, kappa, _ptr(out), _ptr(inp), parity, int(inverse), prec, stream))


def bq_dirac_apply(h, out, inp, kappa, csw, prec, recon=BQ_RECON18, stream=None):
    _check(h, lib().bq_dirac_apply(h, _ptr(out), _ptr(inp), kappa, csw, prec, recon, _stream_ptr(stream)))


def bq_schur_apply(h, out, inp, tmp, kappa, csw, prec, recon=BQ_RECON18, stream=None):
    _check(h, lib().bq_schur_apply(h, _ptr(out), _ptr(inp), _ptr(tmp), kappa, csw, prec, recon, _stream_ptr(stream)))


def bq_wilson_apply_multi(h, out, inp, nrhs, kappa, parity, prec=BQ_FP32, recon=BQ_RECON18, stream=None):
    _check(h, lib().bq_wilson_apply_multi(h, _ptr(out), _ptr(inp), nrhs, kappa, parity, prec, recon, _stream_ptr(stream)))


def bq_schur_apply_multi(h, out, inp, tmp, nrhs, kappa, csw, prec, recon=BQ_RECON18, stream=None):
    _check(h, lib().bq_schur_apply_multi(h, _ptr(out), _ptr(inp), _ptr(tmp), nrhs, kappa, csw, prec, recon,
                                         _stream_ptr(stream)))


def bq_dirac_apply_mode(h, out, inp, tmp, kappa, csw, mode, prec, recon=BQ_RECON18, stream=None):
    _check(h, lib().bq_dirac_apply_mode(h, _ptr(out), _ptr(inp), _ptr(tmp), kappa, csw, mode, prec, recon, _stream_ptr(stream)))


def bq_schur_apply_mode(h, out, inp, tmp, tmp2, kappa, csw, mode, prec, recon=BQ_RECON18, stream=None):
    _check(h, lib().bq_schur_apply_mode(h, _ptr(out), _ptr(inp), _ptr(tmp), _ptr(tmp2), kappa, csw, mode, prec, recon,
                                        _stream_ptr(stream)))


def bq_schur_apply_dots(h, out, inp, tmp, kappa, csw, prec, recon=BQ_RECON18, w=None):
    """out = M^ inp with the inner products fused into the hop epilogue: w given -> <w,out>; else (<out,inp>, <out,out>)."""
    r = (ctypes.c_double * 3)()
    _check(h, lib().bq_schur_apply_dots(h, _ptr(out), _ptr(inp), _ptr(tmp), kappa, csw, prec, recon, _ptr(w), r))
    if w is not None:
        return complex(r[0], r[1])
    return complex(r[0], r[1]), r[2]


def bq_solve(h, b, x, kappa, tol, opts: bq_solve_opts | None = None, raise_on_fail=True):
    """b, x: canonical complex128 arrays (numpy host arrays or torch CUDA tensors); x is in/out.  Returns bq_solve_info."""
    info = bq_solve_info()
    st = lib().bq_solve(h, _canonical(h, b, 1, "b"), _canonical(h, x, 1, "x"), kappa, tol, ctypes.byref(opts) if opts is not None else None,
                        ctypes.byref(info))
    _check(h, st, allow=() if raise_on_fail else (BQ_ENOTCONVERGED, BQ_EBREAKDOWN))
    return info


def bq_solve_multi(h, b, x, nrhs, kappa, tol, opts: bq_solve_opts | None = None, raise_on_fail=True):
    """b, x: [nrhs, Lt,Lz,Ly,Lx,4,3] complex128 (numpy host arrays or torch CUDA tensors); x is in/out.  Returns [bq_solve_info]."""
    if nrhs < 1:
        raise BqError(BQ_EINVAL, "bq_solve_multi: nrhs must be >= 1")
    infos = (bq_solve_info * nrhs)()
    st = lib().bq_solve_multi(h, _canonical(h, b, nrhs, "b"), _canonical(h, x, nrhs, "x"), nrhs, kappa, tol,
                              ctypes.byref(opts) if opts is not None else None, infos)
    _check(h, st, allow=() if raise_on_fail else (BQ_ENOTCONVERGED, BQ_EBREAKDOWN))
    return list(infos)


def bq_propagator(h, src_site, S, kappa, tol, opts: bq_solve_opts | None = None, raise_on_fail=True):
    """S: [12, Lt,Lz,Ly,Lx,4,3] complex128 output (numpy host array or torch CUDA tensor); src_site = (x, y, z, t)."""
    infos = (bq_solve_info * 12)()
    site = (_i * 4)(*[int(v) for v in src_site])
    st = lib().bq_propagator(h, site, _canonical(h, S, 12, "S"), kappa, tol, ctypes.byref(opts) if opts is not None else None, infos)
    _check(h, st, allow=() if raise_on_fail else (BQ_ENOTCONVERGED, BQ_EBREAKDOWN))
    return list(infos)


def bq_get_counters(h):
    """{'launches': all kernels, 'hop_fp64' / 'hop_fp32' / 'hop_half': hop applications per right-hand side,
    'ls': launches of the link-stationary multi-rhs kernels, 'lsp': of those, direct launches of the direction-split one, 'idle_*': hop applications that returned at entry because
    their right-hand side had already converged (useful = hop_* - idle_*)} since handle creation."""
    out = (ctypes.c_ulonglong * 9)()
    _check(h, lib().bq_get_counters(h, out))
    return {"launches": out[0], "hop_fp64": out[1], "hop_fp32": out[2], "hop_half": out[3], "ls": out[4],
            "idle_fp64": out[5], "idle_fp32": out[6], "idle_half": out[7], "lsp": out[8]}


BQ_K = {"hop": 0, "hop_xpay": 1, "hop_clovinv": 2, "hop_clov_xpay": 3, "schur": 4, "norm2": 5, "p_update": 6, "alpha": 7,
        "s_update": 8, "omega": 9, "final": 10, "bicg_iter": 11, "hop_xpay_alpha": 12, "hop_xpay_omega": 13,
        "bicg_iter_unfused": 14}


def bq_bench_kernel(h, which, prec, recon=BQ_RECON18, csw=0.0, kappa=0.125, reps=200, nsets=3):
    """(microseconds per launch, algorithmic bytes per launch) of one internal kernel (bq_kernel_id or its name)."""
    us, nb = ctypes.c_double(0), ctypes.c_double(0)
    _check(h, lib().bq_bench_kernel(h, BQ_K[which] if isinstance(which, str) else which, prec, recon, csw, kappa, reps, nsets,
                                    ctypes.byref(us), ctypes.byref(nb)))
    return us.value, nb.value


def bq_bench_kernel_multi(h, which, prec, nrhs, recon=BQ_RECON18, csw=0.0, kappa=0.125, reps=50, nsets=2):
    """(microseconds per launch, algorithmic bytes per launch) of one multi-rhs kernel; a launch covers nrhs fields."""
    us, nb = ctypes.c_double(0), ctypes.c_double(0)
    _check(h, lib().bq_bench_kernel_multi(h, BQ_K[which] if isinstance(which, str) else which, prec, recon, csw, kappa, nrhs,
                                          reps, nsets, ctypes.byref(us), ctypes.byref(nb)))
    return us.value, nb.value


def bq_blas_norm2(h, a, prec):
    r = ctypes.c_double(0)
    _check(h, lib().bq_blas_norm2(h, _ptr(a), prec, ctypes.byref(r)))
    return r.value


def bq_field_norm2_noalloc(a, nsites, prec, result, stream=None):
    """|a|^2 of an internal-layout field of nsites sites into `result` (one float64 on the device) — the entry point for
    callers that must not allocate device memory (include/bq.h): no handle, no workspace; its scratch is a fixed array
    inside libbq.so.  Nothing is synchronised: read `result` once the stream has got there."""
    err = ctypes.create_string_buffer(512)
    st = lib().bq_field_norm2_noalloc(_ptr(a), int(nsites), prec, _ptr(result), _stream_ptr(stream), err, len(err))
    if st != BQ_OK:
        raise BqError(st, f"{lib().bq_status_string(st).decode()}: {err.value.decode()}")


def bq_blas_cdot(h, a, b, prec):
    r = (ctypes.c_double * 2)()
    _check(h, lib().bq_blas_cdot(h, _ptr(a), _ptr(b), prec, r))
    return complex(r[0], r[1])


def bq_blas_caxpy(h, alpha, x, y, prec):
    a = (ctypes.c_double * 2)(complex(alpha).real, complex(alpha).imag)
    _check(h, lib().bq_blas_caxpy(h, a, _ptr(x), _ptr(y), prec))


def bq_blas_bicg_update(h, alpha, omega, p, s, t, rhat, x, r, prec):
    a = (ctypes.c_double * 2)(complex(alpha).real, complex(alpha).imag)
    w = (ctypes.c_double * 2)(complex(omega).real, complex(omega).imag)
    r2 = ctypes.c_double(0)
    rr = (ctypes.c_double * 2)()
    _check(h, lib().bq_blas_bicg_update(h, a, w, _ptr(p), _ptr(s), _ptr(t), _ptr(rhat), _ptr(x), _ptr(r), prec,
                                        ctypes.byref(r2), rr))
    return r2.value, complex(rr[0], rr[1])


# ---- domain decomposition (opt-in; include/bq.h) -------------------------------------------
def _ptr_array(items):
    arr = (_vp * len(items))()
    for k, it in enumerate(items):
        arr[k] = it.value if hasattr(it, "value") else _ptr(it)
    return arr


def bq_lattice_create_sub(lx, ly, lz, lt, grid, coords, bc_phase=None):
    h = _vp()
    bc = None
    if bc_phase is not None:
        arr = np.asarray(bc_phase, dtype=np.complex128).view(np.float64)
        bc = (ctypes.c_double * 8)(*arr)
    st = lib().bq_lattice_create_sub(lx, ly, lz, lt, bc, (_i * 4)(*[int(v) for v in grid]), (_i * 4)(*[int(v) for v in coords]),
                                     ctypes.byref(h))
    if st != BQ_OK:
        raise BqError(st, lib().bq_status_string(st).decode())
    _DIMS[h.value] = (int(lx), int(ly), int(lz), int(lt))
    return h


def bq_dd_face_bytes(h, mu, prec):
    n = ctypes.c_size_t(0)
    _check(h, lib().bq_dd_face_bytes(h, mu, prec, ctypes.byref(n)))
    return n.value


def bq_dd_pack(h, send, inp, out_parity, prec, recon=BQ_RECON18, stream=None):
    """send: 8 buffers (or None for unpartitioned directions), index 2*mu + side."""
    _check(h, lib().bq_dd_pack(h, _ptr_array(send), _ptr(inp), out_parity, prec, recon, _stream_ptr(stream)))


def bq_dd_unpack(h, out, recv, scale, out_parity, prec, recon=BQ_RECON18, stream=None):
    _check(h, lib().bq_dd_unpack(h, _ptr(out), _ptr_array(recv), scale, out_parity, prec, recon, _stream_ptr(stream)))


def bq_dd_wilson_apply(handles, outs, ins, kappa, parity, prec, recon=BQ_RECON18, stream=None):
    """Virtual ranks: handles[r], outs[r], ins[r] for every rank r of the grid (rank number: x fastest)."""
    _check(handles[0], lib().bq_dd_wilson_apply(_ptr_array(handles), len(handles), _ptr_array(outs), _ptr_array(ins), kappa, parity, prec,
                                                recon, _stream_ptr(stream)))


def bq_dd_solve(handles, bs, xs, kappa, tol, max_iter=0, raise_on_fail=True):
    """bs[r], xs[r]: the local canonical complex128 blocks of rank r (numpy host arrays or torch CUDA tensors); xs is in/out."""
    info = bq_solve_info()
    st = lib().bq_dd_solve(_ptr_array(handles), len(handles), _ptr_array([_canonical(h, b, 1, "b") for h, b in zip(handles, bs)]),
                           _ptr_array([_canonical(h, x, 1, "x") for h, x in zip(handles, xs)]), kappa, tol, max_iter, ctypes.byref(info))
    _check(handles[0], st, allow=() if raise_on_fail else (BQ_ENOTCONVERGED, BQ_EBREAKDOWN))
    return info


# ---- convenience wrapper: owns the handle and allocates internal-layout buffers with torch --------------
class Lattice:
    """RAII handle + torch-allocated internal-layout fields.  Pure marshalling; no arithmetic."""

    def __init__(self, L, bc_phase=None, grid=None, coords=None):
        """grid / coords given: the sub-lattice of one rank of a process grid (L = local extents; opt-in domain decomposition)."""
        self.L = tuple(int(v) for v in L)
        self.h = bq_lattice_create(*self.L, bc_phase) if grid is None else bq_lattice_create_sub(*self.L, grid, coords, bc_phase)

    def close(self):
        if self.h is not None:
            bq_lattice_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def field(self, prec, parity=BQ_EVEN):
        import torch
        return torch.zeros(bq_field_bytes(self.h, prec, parity), dtype=torch.uint8, device="cuda")

    def import_field(self, canonical, prec, parity):
        """canonical: complex128 numpy array [Lt,Lz,Ly,Lx,4,3] or torch CUDA tensor -> internal-layout buffer."""
        import torch
        if isinstance(canonical, np.ndarray):
            canonical = torch.from_numpy(np.ascontiguousarray(canonical, dtype=np.complex128)).cuda()
        buf = self.field(prec, parity)
        bq_field_import(self.h, buf, canonical, parity, prec)
        return buf

    def export_field(self, internal, prec, parity):
        """internal-layout buffer -> complex128 numpy array of the whole lattice (other parity zero)."""
        import torch
        Lx, Ly, Lz, Lt = self.L
        out = torch.zeros((Lt, Lz, Ly, Lx, 4, 3), dtype=torch.complex128, device="cuda")
        bq_field_export(self.h, out, internal, parity, prec)
        return out.cpu().numpy()
