"""GPU parity: the CUDA path (through the C-ABI, libbq.so) against the CPU oracle, element by element.

Thresholds (BASELINE.json north_star; SURVEY.md §8(c) acceptance (i)): max-norm relative error per applied
operator 1e-12 fp64, 1e-5 fp32, 5e-3 half storage, the low-precision runs fed the rounded copy of the same
fp64 inputs and compared with the oracle on the UN-rounded inputs.
"""
import numpy as np
import pytest

from oracle import bqo
from paper_2111_04457_b200 import inputs
from tests.conftest import relmax

pytestmark = pytest.mark.gpu

TOL = {0: 1e-12, 1: 1e-5, 2: 5e-3}
PRECS = [0, 1, 2]
RECONS = [0, 1]
# several 128-thread tiles with a ragged tail (Vh = 8*4*6*4/2 = 384 = 3 tiles; 6*6*4*10/2 = 720 = 5.6 tiles), an L = 2 direction
LATTICES = [(4, 4, 4, 4), (8, 4, 6, 4), (6, 6, 4, 10), (2, 2, 2, 2), (4, 2, 6, 2)]
GENERAL_BC = np.exp(1j * np.array([0.4, -1.3, 2.0, 0.9]))


@pytest.fixture(scope="module")
def bq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2111_04457_b200 import bq as _bq
    _bq.lib()   # fails loudly if libbq.so is missing
    return _bq


def make_case(L, seed, eps):
    return inputs.gauge(L, seed, eps), inputs.spinor(L, seed)


# ---------------------------------------------------------------------------------------------------
# A1: import / export
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", LATTICES)
def test_import_export_roundtrip_fp64_bit_exact(bq, L):
    psi = inputs.spinor(L, 11)
    par = inputs.site_parity(L)
    with bq.Lattice(L) as lat:
        full = lat.import_field(psi, bq.BQ_FP64, bq.BQ_FULL)
        assert np.array_equal(lat.export_field(full, bq.BQ_FP64, bq.BQ_FULL), psi)
        for p in (0, 1):
            buf = lat.import_field(psi, bq.BQ_FP64, p)
            back = lat.export_field(buf, bq.BQ_FP64, p)
            assert np.array_equal(back, np.where((par == p)[..., None, None], psi, 0))


def test_import_rounding_fp32_and_half(bq):
    L = (4, 4, 4, 4)
    psi = inputs.spinor(L, 12)
    psi[0, 0, 0, 0] = 0                       # an all-zero site: norm 0, mantissas 0
    psi[1, 2, 3, 1] *= 1e-3                   # a small site keeps its relative precision thanks to the site norm
    with bq.Lattice(L) as lat:
        b32 = lat.export_field(lat.import_field(psi, bq.BQ_FP32, bq.BQ_FULL), bq.BQ_FP32, bq.BQ_FULL)
        assert np.array_equal(b32, psi.astype(np.complex64).astype(np.complex128))   # round to nearest even
        b16 = lat.export_field(lat.import_field(psi, bq.BQ_HALF, bq.BQ_FULL), bq.BQ_HALF, bq.BQ_FULL)
        # expected by definition (reading S11): n = fp32(max|v_i|), v_i -> fp16(v_i/n) * n
        flat = psi.reshape(-1, 12).view(np.float64).reshape(-1, 24)
        n = np.abs(flat).max(axis=1).astype(np.float32)
        with np.errstate(divide="ignore", invalid="ignore"):
            m = np.where(n[:, None] > 0, flat / n[:, None].astype(np.float64), 0.0).astype(np.float32).astype(np.float16)
        expect = (m.astype(np.float32) * n[:, None]).astype(np.float64).view(np.complex128).reshape(psi.shape)
        assert np.array_equal(b16, expect)
        assert np.all(b16[0, 0, 0, 0] == 0)
        site_err = np.abs(b16 - psi).reshape(-1, 12).max(axis=1) / np.maximum(np.abs(flat).max(axis=1), 1e-300)
        assert site_err.max() < 2.0 ** -11 * 1.01


# ---------------------------------------------------------------------------------------------------
# A3: even-odd hop, every (precision, recon), several geometries and boundary phases
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", LATTICES)
@pytest.mark.parametrize("prec", PRECS)
@pytest.mark.parametrize("recon", RECONS)
def test_hop_parity(bq, L, prec, recon):
    kappa = 0.125
    U, psi = make_case(L, 21, 0.5)
    for bc in (None, GENERAL_BC):
        with bq.Lattice(L, bc) as lat:
            bq.bq_gauge_load(lat.h, U)
            for p in (0, 1):
                ref = bqo.hop_restricted(U, psi, kappa, p, bc=bc)
                src = lat.import_field(psi, prec, 1 - p)
                out = lat.field(prec, p)
                bq.bq_wilson_apply(lat.h, out, src, kappa, p, prec, recon)
                got = lat.export_field(out, prec, p)
                assert relmax(got, ref) < TOL[prec], (L, prec, recon, p)
                mask = (inputs.site_parity(L) == p)[..., None, None]
                assert np.all(got[~np.broadcast_to(mask, got.shape)] == 0)


@pytest.mark.parametrize("L", [(8, 8, 8, 8), (6, 6, 4, 10)])
@pytest.mark.parametrize("recon", RECONS)
def test_small_lattice_build_of_the_fp32_hop(bq, L, recon, monkeypatch):
    """On lattices whose CTAs are all resident at once the fp32 hop runs an uncapped-register build of the same kernel
    (hop_kernel<..., SMALL>; BQ_HOP_SMALL is read when the handle is made).  Both builds against the oracle, and bit for bit against each
    other: plain hop, xpay / clover epilogues through the Schur operator with its fused inner products."""
    import torch
    kappa, csw = 0.125, 1.0
    U, psi = make_case(L, 23, 0.5)
    ref = bqo.hop_restricted(U, psi, kappa, 0)
    outs = {}
    for small in ("0", "1000000"):
        monkeypatch.setenv("BQ_HOP_SMALL", small)
        with bq.Lattice(L) as lat:
            bq.bq_gauge_load(lat.h, U)
            src = lat.import_field(psi, bq.BQ_FP32, bq.BQ_ODD)
            out = lat.field(bq.BQ_FP32, bq.BQ_EVEN)
            bq.bq_wilson_apply(lat.h, out, src, kappa, bq.BQ_EVEN, bq.BQ_FP32, recon)
            assert relmax(lat.export_field(out, bq.BQ_FP32, bq.BQ_EVEN), ref) < TOL[bq.BQ_FP32], (L, recon, small)
            src_e = lat.import_field(psi, bq.BQ_FP32, bq.BQ_EVEN)
            res = [out.clone()]
            for c in (0.0, csw):
                o, tmp = lat.field(bq.BQ_FP32, bq.BQ_EVEN), lat.field(bq.BQ_FP32, bq.BQ_EVEN)
                d1 = bq.bq_schur_apply_dots(lat.h, o, src_e, tmp, kappa, c, bq.BQ_FP32, recon, src_e)        # <w, out>
                d2, d3 = bq.bq_schur_apply_dots(lat.h, o, src_e, tmp, kappa, c, bq.BQ_FP32, recon)           # <out, in>, <out, out>
                res += [o.clone(), torch.tensor([d1.real, d1.imag, d2.real, d2.imag, d3], dtype=torch.float64)]
            outs[small] = res
    for x, y in zip(outs["0"], outs["1000000"]):
        assert torch.equal(x, y)


@pytest.mark.parametrize("prec", PRECS)
@pytest.mark.parametrize("recon", RECONS)
def test_full_wilson_apply(bq, prec, recon):
    L = (8, 4, 6, 4)
    kappa = 0.12
    U, psi = make_case(L, 22, 0.3)
    ref = bqo.dirac_apply(U, psi, kappa)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        src = lat.import_field(psi, prec, bq.BQ_FULL)
        out = lat.field(prec, bq.BQ_FULL)
        bq.bq_wilson_apply(lat.h, out, src, kappa, bq.BQ_FULL, prec, recon)
        assert relmax(lat.export_field(out, prec, bq.BQ_FULL), ref) < TOL[prec]


def test_config1_apply_fp64(bq, cfg1):
    """BASELINE.json config 1: 4^4, fp64, kappa = 0.12, apply D once."""
    ref = bqo.dirac_apply(cfg1["U"], cfg1["b"], cfg1["kappa"])
    with bq.Lattice(cfg1["L"]) as lat:
        bq.bq_gauge_load(lat.h, cfg1["U"])
        src = lat.import_field(cfg1["b"], bq.BQ_FP64, bq.BQ_FULL)
        out = lat.field(bq.BQ_FP64, bq.BQ_FULL)
        bq.bq_wilson_apply(lat.h, out, src, cfg1["kappa"], bq.BQ_FULL, bq.BQ_FP64, bq.BQ_RECON18)
        assert relmax(lat.export_field(out, bq.BQ_FP64, bq.BQ_FULL), ref) < 1e-12


def test_hop_is_deterministic_and_gauge_from_device(bq):
    """Repeated applies are bitwise identical (reading S12); a device-resident U gives the same result as a host U."""
    import torch
    L = (8, 8, 4, 4)
    U, psi = make_case(L, 23, 0.3)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        src = lat.import_field(psi, bq.BQ_FP32, bq.BQ_ODD)
        out1, out2 = lat.field(bq.BQ_FP32, bq.BQ_EVEN), lat.field(bq.BQ_FP32, bq.BQ_EVEN)
        bq.bq_wilson_apply(lat.h, out1, src, 0.125, bq.BQ_EVEN)
        for _ in range(20):
            bq.bq_wilson_apply(lat.h, out2, src, 0.125, bq.BQ_EVEN)
        assert torch.equal(out1, out2)
        bq.bq_gauge_load(lat.h, torch.from_numpy(U).cuda())
        bq.bq_wilson_apply(lat.h, out2, src, 0.125, bq.BQ_EVEN)
        assert torch.equal(out1, out2)


def test_hop_on_user_stream(bq):
    import torch
    L = (4, 4, 4, 4)
    U, psi = make_case(L, 24, 0.3)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        src = lat.import_field(psi, bq.BQ_FP32, bq.BQ_ODD)
        a, b = lat.field(bq.BQ_FP32, bq.BQ_EVEN), lat.field(bq.BQ_FP32, bq.BQ_EVEN)
        bq.bq_wilson_apply(lat.h, a, src, 0.125, bq.BQ_EVEN)
        torch.cuda.synchronize()
        st = torch.cuda.Stream()
        bq.bq_wilson_apply(lat.h, b, src, 0.125, bq.BQ_EVEN, stream=st)
        st.synchronize()
        assert torch.equal(a, b)


# ---------------------------------------------------------------------------------------------------
# A4 / A5: clover
# ---------------------------------------------------------------------------------------------------
CLOVER_TOL = {0: 1e-12, 1: 1e-5, 2: 5e-3}


@pytest.mark.parametrize("prec", PRECS)
def test_clover_apply_and_inverse(bq, prec):
    L = (4, 6, 4, 4)
    csw, kappa = 1.0, 0.1215
    U, psi = make_case(L, 31, 0.5)
    A = bqo.clover_build(U, csw, kappa)
    Ainv = bqo.site_matrix_invert(A)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        bq.bq_clover_apply(lat.h, csw, kappa, None, None, bq.BQ_FULL, 0, prec)      # build only
        src = lat.import_field(psi, prec, bq.BQ_FULL)
        out = lat.field(prec, bq.BQ_FULL)
        for inverse, ref in ((0, bqo.site_matrix_apply(A, psi)), (1, bqo.site_matrix_apply(Ainv, psi))):
            bq.bq_clover_apply(lat.h, csw, kappa, out, src, bq.BQ_FULL, inverse, prec)
            assert relmax(lat.export_field(out, prec, bq.BQ_FULL), ref) < CLOVER_TOL[prec], (prec, inverse)
        # one parity, in place
        par = inputs.site_parity(L)
        for p in (0, 1):
            buf = lat.import_field(psi, prec, p)
            bq.bq_clover_apply(lat.h, csw, kappa, buf, buf, p, 0, prec)
            ref = np.where((par == p)[..., None, None], bqo.site_matrix_apply(A, psi), 0)
            assert relmax(lat.export_field(buf, prec, p), ref) < CLOVER_TOL[prec]


@pytest.mark.parametrize("prec", PRECS)
@pytest.mark.parametrize("recon", RECONS)
def test_wilson_clover_dirac_and_schur(bq, prec, recon):
    L = (4, 4, 6, 8)
    csw, kappa = 1.0, 0.1215
    U, psi = make_case(L, 32, 0.5)
    A = bqo.clover_build(U, csw, kappa)
    Ainv = bqo.site_matrix_invert(A)
    even = (inputs.site_parity(L) == 0)[..., None, None]
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        src = lat.import_field(psi, prec, bq.BQ_FULL)
        out = lat.field(prec, bq.BQ_FULL)
        bq.bq_dirac_apply(lat.h, out, src, kappa, csw, prec, recon)
        assert relmax(lat.export_field(out, prec, bq.BQ_FULL), bqo.dirac_apply(U, psi, kappa, A=A)) < TOL[prec]
        # Schur complement, clover and Wilson
        xe = lat.import_field(psi, prec, bq.BQ_EVEN)
        o, tmp = lat.field(prec, bq.BQ_EVEN), lat.field(prec, bq.BQ_ODD)
        bq.bq_schur_apply(lat.h, o, xe, tmp, kappa, csw, prec, recon)
        ref = bqo.schur_apply(U, np.where(even, psi, 0), kappa, A=A, Ainv=Ainv)
        assert relmax(lat.export_field(o, prec, bq.BQ_EVEN), ref) < 2 * TOL[prec]     # two hops
        bq.bq_schur_apply(lat.h, o, xe, tmp, kappa, 0.0, prec, recon)
        ref = bqo.schur_apply(U, np.where(even, psi, 0), kappa)
        assert relmax(lat.export_field(o, prec, bq.BQ_EVEN), ref) < 2 * TOL[prec]


@pytest.mark.parametrize("prec", PRECS)
@pytest.mark.parametrize("csw", [0.0, 1.0])
@pytest.mark.parametrize("L", [(4, 4, 6, 8), (6, 6, 4, 10)])
def test_schur_fused_inner_products(bq, prec, csw, L):
    """A6 (iii), (v) fused into the hop epilogue: <w, M^x>, <M^x, x>, <M^x, M^x> against the oracle's operator and
    numpy sums; the output field itself must equal the unfused bq_schur_apply (bit for bit in fp64 / fp32; in half
    storage the two kernel instantiations may contract `z*n + acc` differently, so there to one fp16 ulp)."""
    import torch
    kappa = 0.1215
    U, psi = make_case(L, 34, 0.5)
    wv = inputs.spinor(L, 35)
    even = (inputs.site_parity(L) == 0)[..., None, None]
    A = bqo.clover_build(U, csw, kappa) if csw else None
    Ainv = bqo.site_matrix_invert(A) if csw else None
    xe_ref, w_ref = np.where(even, psi, 0), np.where(even, wv, 0)
    ref = bqo.schur_apply(U, xe_ref, kappa, A=A, Ainv=Ainv)
    # storage-rounding bound of an inner product, relative to |a||b|
    tol = {0: 1e-13, 1: 2e-6, 2: 2e-3}[prec]
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        xe = lat.import_field(psi, prec, bq.BQ_EVEN)
        we = lat.import_field(wv, prec, bq.BQ_EVEN)
        o, o2, tmp = lat.field(prec, bq.BQ_EVEN), lat.field(prec, bq.BQ_EVEN), lat.field(prec, bq.BQ_ODD)
        bq.bq_schur_apply(lat.h, o2, xe, tmp, kappa, csw, prec)
        nr, nx, nw = np.linalg.norm(ref), np.linalg.norm(xe_ref), np.linalg.norm(w_ref)
        unfused = lat.export_field(o2, prec, bq.BQ_EVEN)

        def same_field():
            if prec != 2:
                return torch.equal(o, o2)
            return relmax(lat.export_field(o, prec, bq.BQ_EVEN), unfused) < 2.0 ** -10

        for rep in range(2):    # twice: no state may be left behind by the first launch
            wd = bq.bq_schur_apply_dots(lat.h, o, xe, tmp, kappa, csw, prec, w=we)
            assert same_field()
            assert abs(wd - np.vdot(w_ref, ref)) < tol * nw * nr
            ts, tt = bq.bq_schur_apply_dots(lat.h, o, xe, tmp, kappa, csw, prec)
            assert same_field()
            assert abs(ts - np.vdot(ref, xe_ref)) < tol * nr * nx
            assert abs(tt - np.vdot(ref, ref).real) < tol * nr * nr
            if rep == 0:
                first = (wd, ts, tt)
            else:
                assert first == (wd, ts, tt)      # fixed summation order: bitwise reproducible


def test_clover_rebuilds_on_new_gauge_or_parameters(bq):
    L = (4, 4, 4, 4)
    psi = inputs.spinor(L, 33)
    with bq.Lattice(L) as lat:
        for seed, csw, kappa in ((1, 1.0, 0.12), (2, 1.0, 0.12), (2, 1.7, 0.11)):
            U = inputs.gauge(L, seed, 0.5)
            bq.bq_gauge_load(lat.h, U)
            src = lat.import_field(psi, bq.BQ_FP64, bq.BQ_FULL)
            out = lat.field(bq.BQ_FP64, bq.BQ_FULL)
            bq.bq_clover_apply(lat.h, csw, kappa, out, src, bq.BQ_FULL, 0, bq.BQ_FP64)
            ref = bqo.site_matrix_apply(bqo.clover_build(U, csw, kappa), psi)
            assert relmax(lat.export_field(out, bq.BQ_FP64, bq.BQ_FULL), ref) < 1e-12


def test_singular_clover_is_reported(bq):
    L = (4, 4, 4, 4)
    U = inputs.gauge(L, 34, 0.7)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        with pytest.raises(bq.BqError) as e:
            bq.bq_clover_apply(lat.h, 40.0, 0.2, None, None, bq.BQ_FULL, 0, bq.BQ_FP64)   # csw*kappa*|F| >> 1
        assert e.value.status == bq.BQ_ESINGULAR_CLOVER


# ---------------------------------------------------------------------------------------------------
# error behaviour on the device
# ---------------------------------------------------------------------------------------------------
def test_errors(bq):
    with bq.Lattice((4, 4, 4, 4)) as lat:
        a, b = lat.field(bq.BQ_FP32, 0), lat.field(bq.BQ_FP32, 1)
        with pytest.raises(bq.BqError) as e:
            bq.bq_wilson_apply(lat.h, a, b, 0.1, 0)
        assert e.value.status == bq.BQ_ENOGAUGE
        bq.bq_gauge_load(lat.h, inputs.unit_gauge((4, 4, 4, 4)))
        for args in ((a, a, 0.1, 0), (a, b, 0.1, 7), (None, b, 0.1, 0)):
            with pytest.raises(bq.BqError) as e:
                bq.bq_wilson_apply(lat.h, *args)
            assert e.value.status == bq.BQ_EINVAL
        with pytest.raises(bq.BqError) as e:
            bq.bq_wilson_apply(lat.h, a, b, 0.1, 0, 5, 0)
        assert e.value.status == bq.BQ_EINVAL
        assert bq.bq_field_bytes(lat.h, bq.BQ_HALF, bq.BQ_FULL) == 2 * 128 * 52
        assert bq.bq_field_bytes(lat.h, bq.BQ_FP64, bq.BQ_EVEN) == 128 * 192
