"""bq_field_norm2_noalloc (include/bq.h) — the squared norm for programs that cannot allocate device memory.

Some users of libbq.so run inside a host that owns all of the GPU's memory through an allocator of its own (a framework's
caching allocator, a server with a fixed arena), or next to a thread that is capturing a stream in the global capture mode,
or in a monitoring loop that must not stall the device: a cudaMalloc from this library would fail, break the capture or
synchronise the GPU.  The handle-based reductions all allocate a workspace on first use; this entry point does not — its
scratch (per-block partial sums and an arrival counter) is a fixed 128 KiB array compiled into the library, shared by all
calls on a device, and the field size is capped at BQ_NOALLOC_MAX_SITES accordingly.

What is checked: the new call against the existing handle-based path (bq_blas_norm2) on the same stored field, within the
tolerance tests/test_gpu_solver.py uses for that path, on consecutive calls that reuse the shared scratch (a stale partial
sum or arrival counter from the first call would corrupt the second); that the calls leave the amount of free device
memory unchanged; and that a field beyond the cap is refused with a message instead of overrunning the array.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It does not depend on anything the other tests leave behind (it passes alone in a fresh process as well).
"""
import numpy as np
import pytest

from paper_2111_04457_b200 import inputs

MAX_SITES = 16384 * 1024          # BQ_NOALLOC_MAX_SITES
REL_TOL = {0: 1e-13, 1: 1e-6, 2: 1e-6}   # as test_blas_reductions_and_axpy: both paths sum the same stored numbers


@pytest.fixture(scope="module")
def bq():
    from paper_2111_04457_b200 import build
    build.build()
    from paper_2111_04457_b200 import bq as _bq
    _bq.lib()
    return _bq


@pytest.mark.gpu
@pytest.mark.parametrize("prec", [0, 1, 2])
@pytest.mark.parametrize("L", [(8, 6, 6, 10), (16, 12, 10, 10)])     # 1440 and 9600 sites per parity: 2 and 10 blocks, ragged last block
def test_matches_handle_based_norm_on_consecutive_calls(bq, prec, L):
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    V = int(np.prod(L))
    a = inputs.spinor(L, 71)
    b = 3.0 * inputs.spinor(L, 72, inputs.STREAM_TEST)      # another norm, so that a result left over from call 1 cannot pass call 2
    with bq.Lattice(L) as lat:
        # one-parity fields and a full-lattice ([even | odd]) field
        da = lat.import_field(a, prec, bq.BQ_EVEN)
        db = lat.import_field(b, prec, bq.BQ_ODD)
        dfull = lat.import_field(a, prec, bq.BQ_FULL)
        per_parity = bq.bq_field_bytes(lat.h, prec, bq.BQ_EVEN)
        want_a = bq.bq_blas_norm2(lat.h, da, prec)           # the existing path (allocates its workspace here)
        want_b = bq.bq_blas_norm2(lat.h, db, prec)
        want_full = want_a + bq.bq_blas_norm2(lat.h, dfull[per_parity:], prec)
        assert want_a > 0 and want_b > 2 * want_a

        out = torch.full((4,), -1.0, dtype=torch.float64, device="cuda")    # the caller's outputs; nothing below allocates
        bq.bq_field_norm2_noalloc(da, V // 2, prec, out[0:1])               # first call on the device also does the set-up
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        bq.bq_field_norm2_noalloc(db, V // 2, prec, out[1:2])               # back to back, same stream, same scratch
        bq.bq_field_norm2_noalloc(dfull, V, prec, out[2:3])
        bq.bq_field_norm2_noalloc(da, V // 2, prec, out[3:4])
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the amount of free device memory"
        got = out.cpu().numpy()
        assert abs(got[0] - want_a) <= REL_TOL[prec] * want_a
        assert abs(got[1] - want_b) <= REL_TOL[prec] * want_b
        assert abs(got[2] - want_full) <= REL_TOL[prec] * want_full
        assert got[3] == got[0], "fixed summation order: the same field gives the same bits, whatever ran in between"


@pytest.mark.gpu
def test_runs_on_a_side_stream_and_handles_an_empty_field(bq):
    import torch
    L = (8, 8, 8, 8)
    with bq.Lattice(L) as lat:
        da = lat.import_field(inputs.spinor(L, 73), bq.BQ_FP32, bq.BQ_EVEN)
        want = bq.bq_blas_norm2(lat.h, da, bq.BQ_FP32)
        out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        bq.bq_field_norm2_noalloc(da, 2048, bq.BQ_FP32, out[0:1], stream=s)
        bq.bq_field_norm2_noalloc(da, 0, bq.BQ_FP32, out[1:2], stream=s)
        s.synchronize()
        got = out.cpu().numpy()
        assert abs(got[0] - want) <= 1e-6 * want and got[1] == 0.0


def test_refuses_what_the_fixed_scratch_cannot_cover(bq):
    """Validation comes before any device work, so this runs without a GPU: the pointers are never dereferenced."""
    fake_field, fake_result = 4096, 8192
    with pytest.raises(bq.BqError) as e:
        bq.bq_field_norm2_noalloc(fake_field, MAX_SITES + 8, bq.BQ_FP32, fake_result)
    assert e.value.status == bq.BQ_EINVAL and "BQ_NOALLOC_MAX_SITES" in str(e.value)
    for bad_sites in (-8, 12):                       # the layout's tiles hold 8 sites
        with pytest.raises(bq.BqError) as e:
            bq.bq_field_norm2_noalloc(fake_field, bad_sites, bq.BQ_FP32, fake_result)
        assert e.value.status == bq.BQ_EINVAL
    with pytest.raises(bq.BqError) as e:
        bq.bq_field_norm2_noalloc(fake_field + 4, 8, bq.BQ_FP32, fake_result)      # misaligned field
    assert e.value.status == bq.BQ_EINVAL
    with pytest.raises(bq.BqError) as e:
        bq.bq_field_norm2_noalloc(fake_field, 8, 7, fake_result)                   # no such precision
    assert e.value.status == bq.BQ_EINVAL
    with pytest.raises(bq.BqError) as e:
        bq.bq_field_norm2_noalloc(None, 8, bq.BQ_FP32, fake_result)
    assert e.value.status == bq.BQ_EINVAL
