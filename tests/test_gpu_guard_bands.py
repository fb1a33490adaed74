"""Out-of-bounds write detector (compute-sanitizer is closed on this pool): every output buffer of the kernels with padded
or ragged launch shapes is a window inside a larger allocation filled with a sentinel; after the call the bands on both
sides must be untouched.  Geometries: Vh not a multiple of the CTA size, multi-rhs CTAs padded to whole warps, chunked
batches, the patch mapping."""
import numpy as np
import pytest

from paper_2111_04457_b200 import inputs

pytestmark = pytest.mark.gpu

GUARD = 4096
SENTINEL = 0xAB


@pytest.fixture(scope="module")
def bq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2111_04457_b200 import bq as _bq
    _bq.lib()
    return _bq


class Guarded:
    def __init__(self, nbytes):
        import torch
        self.raw = torch.full((nbytes + 2 * GUARD,), SENTINEL, dtype=torch.uint8, device="cuda")
        self.buf = self.raw[GUARD:GUARD + nbytes]
        self.buf.zero_()

    def intact(self):
        return bool((self.raw[:GUARD] == SENTINEL).all()) and bool((self.raw[-GUARD:] == SENTINEL).all())


@pytest.mark.parametrize("L", [(6, 6, 4, 10), (4, 2, 6, 2), (16, 2, 6, 4), (2, 2, 2, 2)])
@pytest.mark.parametrize("prec", [0, 1, 2])
def test_no_write_outside_the_output_fields(bq, L, prec):
    import torch
    U = inputs.gauge(L, 31, 0.5)
    kappa, csw = 0.12, 1.0
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        fb = bq.bq_field_bytes(lat.h, prec, bq.BQ_EVEN)
        for nrhs in (1, 3, 12, 19):
            psis = [inputs.spinor(L, 32 + k) for k in range(nrhs)]
            src = torch.cat([lat.import_field(p, prec, bq.BQ_ODD) for p in psis])
            srce = torch.cat([lat.import_field(p, prec, bq.BQ_EVEN) for p in psis])
            out, tmp = Guarded(nrhs * fb), Guarded(nrhs * fb)
            bq.bq_wilson_apply_multi(lat.h, out.buf, src, nrhs, kappa, bq.BQ_EVEN, prec, nrhs % 2)
            assert out.intact(), ("hop", L, prec, nrhs)
            for c in (0.0, csw):
                bq.bq_schur_apply_multi(lat.h, out.buf, srce, tmp.buf, nrhs, kappa, c, prec)
                assert out.intact() and tmp.intact(), ("schur", L, prec, nrhs, c)
        # single-field entry points
        psi = inputs.spinor(L, 40)
        o1, t1, t2 = Guarded(fb), Guarded(fb), Guarded(fb)
        xe = lat.import_field(psi, prec, bq.BQ_EVEN)
        for mode in (bq.BQ_MODE_D, bq.BQ_MODE_DDAG, bq.BQ_MODE_DDAGD):
            bq.bq_schur_apply_mode(lat.h, o1.buf, xe, t1.buf, t2.buf, kappa, csw, mode, prec)
            assert o1.intact() and t1.intact() and t2.intact(), ("schur_mode", L, prec, mode)
        full = Guarded(2 * fb)
        bq.bq_dirac_apply(lat.h, full.buf, lat.import_field(psi, prec, bq.BQ_FULL), kappa, csw, prec)
        assert full.intact()
        imp = Guarded(2 * fb)
        bq.bq_field_import(lat.h, imp.buf, torch.from_numpy(psi).cuda(), bq.BQ_FULL, prec)
        assert imp.intact()
        Lx, Ly, Lz, Lt = L
        canon = Guarded(Lx * Ly * Lz * Lt * 12 * 16)
        bq.bq_field_export(lat.h, canon.buf, imp.buf, bq.BQ_FULL, prec)
        assert canon.intact()
        # BLAS-1 outputs: y of caxpy; x and r of the BiCGStab update (x is an fp32 field when the storage is half)
        y = Guarded(fb)
        y.buf.copy_(xe)
        bq.bq_blas_caxpy(lat.h, 0.3 - 0.2j, xe, y.buf, prec)
        xprec = bq.BQ_FP32 if prec == bq.BQ_HALF else prec
        xacc, r = Guarded(bq.bq_field_bytes(lat.h, xprec, bq.BQ_EVEN)), Guarded(fb)
        bq.bq_blas_bicg_update(lat.h, 0.5 + 0.1j, 0.4 - 0.3j, xe, y.buf, xe, xe, xacc.buf, r.buf, prec)
        assert y.intact() and xacc.intact() and r.intact(), ("blas", L, prec)
