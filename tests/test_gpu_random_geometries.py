"""GPU parity on seeded random geometries: even extents 2..16 in every direction (L = 2 directions, extents that are not
multiples of the 8-site layout tile, x-rows that hold whole tiles and x-rows that do not), random U(1) boundary phases,
random kappa; the hop, its dagger, the Schur operator and the multi-rhs hop against the oracle in all three precisions."""
import numpy as np
import pytest

from oracle import bqo
from paper_2111_04457_b200 import inputs
from tests.conftest import relmax

pytestmark = pytest.mark.gpu

TOL = {0: 1e-12, 1: 1e-5, 2: 5e-3}


@pytest.fixture(scope="module")
def bq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2111_04457_b200 import bq as _bq
    _bq.lib()
    return _bq


def cases(n):
    rng = np.random.default_rng(20211104457)
    out = []
    while len(out) < n:
        L = tuple(int(v) for v in rng.choice([2, 4, 6, 8, 10, 12, 16], size=4))
        if np.prod(L) > 6000:
            continue
        bc = np.exp(1j * rng.uniform(-np.pi, np.pi, 4))
        if len(out) % 3 == 0:
            bc = np.array([1, 1, 1, -1], dtype=complex)          # the configs' boundary condition (real-phase kernels)
        out.append((L, bc, float(rng.uniform(0.05, 0.124)), int(rng.integers(1, 1 << 30))))
    # x-rows of whole tiles (Lx = 16, 32): the patch mapping of the multi-rhs kernel, with 3..5 right-hand sides
    for L, seed in (((16, 2, 4, 6), 1002), ((16, 6, 2, 4), 1003), ((32, 2, 2, 4), 1004)):
        out.append((L, np.exp(1j * rng.uniform(-np.pi, np.pi, 4)), float(rng.uniform(0.05, 0.124)), seed))
    return out


@pytest.mark.parametrize("L,bc,kappa,seed", cases(12))
def test_random_geometry(bq, L, bc, kappa, seed):
    import torch
    U = inputs.gauge(L, seed, 0.6)
    nrhs = 1 + seed % 5
    psis = [inputs.spinor(L, seed + 7 * k) for k in range(nrhs)]
    psi = psis[0]
    even = (inputs.site_parity(L) == 0)[..., None, None]
    ref_hop = [bqo.hop_restricted(U, p, kappa, 0, bc=bc) for p in psis]
    ref_dag = bqo.dirac_apply_dag(U, psi, kappa, bc=bc)
    ref_schur = bqo.schur_apply(U, np.where(even, psi, 0), kappa, bc=bc)
    with bq.Lattice(L, bc) as lat:
        bq.bq_gauge_load(lat.h, U)
        for prec in (0, 1, 2):
            recon = (seed + prec) % 2
            fb = bq.bq_field_bytes(lat.h, prec, bq.BQ_EVEN)
            src = torch.cat([lat.import_field(p, prec, bq.BQ_ODD) for p in psis])
            out = torch.zeros(nrhs * fb, dtype=torch.uint8, device="cuda")
            bq.bq_wilson_apply_multi(lat.h, out, src, nrhs, kappa, bq.BQ_EVEN, prec, recon)
            one = lat.field(prec, bq.BQ_EVEN)
            for k in range(nrhs):
                assert relmax(lat.export_field(out[k * fb:(k + 1) * fb], prec, bq.BQ_EVEN), ref_hop[k]) < TOL[prec], (L, prec, k)
                bq.bq_wilson_apply(lat.h, one, src[k * fb:(k + 1) * fb], kappa, bq.BQ_EVEN, prec, recon)
                assert torch.equal(one, out[k * fb:(k + 1) * fb])
            full = lat.import_field(psi, prec, bq.BQ_FULL)
            o = lat.field(prec, bq.BQ_FULL)
            bq.bq_dirac_apply_mode(lat.h, o, full, None, kappa, 0.0, bq.BQ_MODE_DDAG, prec, recon)
            assert relmax(lat.export_field(o, prec, bq.BQ_FULL), ref_dag) < TOL[prec], (L, prec, "dag")
            xe = lat.import_field(psi, prec, bq.BQ_EVEN)
            oe, tmp = lat.field(prec, bq.BQ_EVEN), lat.field(prec, bq.BQ_EVEN)
            bq.bq_schur_apply(lat.h, oe, xe, tmp, kappa, 0.0, prec, recon)
            assert relmax(lat.export_field(oe, prec, bq.BQ_EVEN), ref_schur) < 2 * TOL[prec], (L, prec, "schur")
