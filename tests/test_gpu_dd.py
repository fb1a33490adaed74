"""Opt-in domain decomposition: the hop and the even-odd BiCGStab on a process
grid of VIRTUAL RANKS (all sub-lattices on one device, faces moved by device copies) against the oracle on the GLOBAL
lattice.  The face kernels, the interior/boundary split and the per-rank reductions are the ones a process per GPU
would run; only the transport differs."""
import numpy as np
import pytest

from oracle import bqo
from paper_2111_04457_b200 import dd, inputs
from tests.conftest import relmax

pytestmark = pytest.mark.gpu

TOL = {0: 1e-12, 1: 1e-5}
GENERAL_BC = np.exp(1j * np.array([0.4, -1.3, 2.0, 0.9]))


@pytest.fixture(scope="module")
def bq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2111_04457_b200 import bq as _bq
    _bq.lib()
    return _bq


class Ranks:
    """nranks sub-lattice handles of a process grid, each with the local block of the global gauge field."""

    def __init__(self, bq, L, grid, U, bc=None):
        self.bq, self.L, self.grid = bq, L, grid
        self.l = dd.local_extents(L, grid)
        self.n = int(np.prod(grid))
        self.lats = [bq.Lattice(self.l, bc, grid=grid, coords=dd.coords_of(r, grid)) for r in range(self.n)]
        for r, lat in enumerate(self.lats):
            bq.bq_gauge_load(lat.h, dd.local_block(U, L, grid, dd.coords_of(r, grid)))

    def handles(self):
        return [lat.h for lat in self.lats]

    def import_field(self, psi, prec, parity):
        return [lat.import_field(dd.local_block(psi, self.L, self.grid, dd.coords_of(r, self.grid)), prec, parity)
                for r, lat in enumerate(self.lats)]

    def export_field(self, bufs, prec, parity):
        return dd.assemble([lat.export_field(b, prec, parity) for lat, b in zip(self.lats, bufs)], self.L, self.grid)

    def close(self):
        for lat in self.lats:
            lat.close()


# grids: two directions partitioned (the paper's 2 x 1 x 1 x 2 example of the verdict), one direction with extent-2 grid
# (lower and upper neighbour are the same rank), all four partitioned (edge and corner sites belong to several faces)
@pytest.mark.parametrize("L,grid", [((8, 8, 8, 16), (2, 1, 1, 2)), ((8, 8, 4, 4), (1, 2, 1, 1)), ((8, 8, 8, 8), (2, 2, 2, 2)),
                                    ((16, 4, 4, 12), (1, 1, 1, 3))])
@pytest.mark.parametrize("prec", [0, 1])
def test_dd_hop_parity(bq, L, grid, prec):
    import torch
    kappa = 0.125
    U = inputs.gauge(L, 1201, 0.5)
    psi = inputs.spinor(L, 1202)
    for bc in (None, GENERAL_BC):
        for recon in (0, 1):
            R = Ranks(bq, L, grid, U, bc)
            try:
                for p in (0, 1):
                    src = R.import_field(psi, prec, 1 - p)
                    out = [lat.field(prec, p) for lat in R.lats]
                    bq.bq_dd_wilson_apply(R.handles(), out, src, kappa, p, prec, recon)
                    torch.cuda.synchronize()
                    ref = bqo.hop_restricted(U, psi, kappa, p, bc=bc)
                    assert relmax(R.export_field(out, prec, p), ref) < TOL[prec], (L, grid, prec, recon, p)
            finally:
                R.close()


@pytest.mark.parametrize("prec", [0, 1])
def test_dd_full_apply(bq, prec):
    """out = D in on [even | odd] buffers over 2 x 1 x 2 x 1 virtual ranks = the oracle's D on the global lattice."""
    import torch
    L, grid, kappa = (8, 4, 8, 4), (2, 1, 2, 1), 0.12
    U = inputs.gauge(L, 1203, 0.4)
    psi = inputs.spinor(L, 1204)
    R = Ranks(bq, L, grid, U)
    try:
        src = R.import_field(psi, prec, bq.BQ_FULL)
        out = [torch.zeros_like(s) for s in src]
        bq.bq_dd_wilson_apply(R.handles(), out, src, kappa, bq.BQ_FULL, prec)
        torch.cuda.synchronize()
        assert relmax(R.export_field(out, prec, bq.BQ_FULL), bqo.dirac_apply(U, psi, kappa)) < TOL[prec]
    finally:
        R.close()


def test_dd_pack_unpack_by_hand(bq):
    """The three-part hop a process per GPU runs — bq_dd_pack, interior bq_wilson_apply, bq_dd_unpack — with the transport done
    by hand according to dd.face_schedule (device copies between the ranks' buffers) = the oracle."""
    import torch
    L, grid, kappa, prec, p = (8, 4, 4, 8), (2, 1, 1, 2), 0.125, 1, 0
    U = inputs.gauge(L, 1205, 0.5)
    psi = inputs.spinor(L, 1206)
    R = Ranks(bq, L, grid, U)
    try:
        src = R.import_field(psi, prec, 1 - p)
        out = [lat.field(prec, p) for lat in R.lats]
        send, recv = [], []
        for lat in R.lats:
            s, r = [None] * 8, [None] * 8
            for mu in range(4):
                if grid[mu] > 1:
                    n = bq.bq_dd_face_bytes(lat.h, mu, prec) // 4
                    for side in range(2):
                        s[2 * mu + side] = torch.zeros(n, dtype=torch.float32, device="cuda")
                        r[2 * mu + side] = torch.zeros(n, dtype=torch.float32, device="cuda")
            send.append(s); recv.append(r)
        for r, lat in enumerate(R.lats):
            bq.bq_dd_pack(lat.h, send[r], src[r], p, prec)
        for r in range(R.n):
            for mu, sside, dest, rside, source in dd.face_schedule(r, grid):
                recv[dest][2 * mu + (1 - sside)].copy_(send[r][2 * mu + sside])     # our side s lands in dest's recv side 1 - s
        for r, lat in enumerate(R.lats):
            bq.bq_wilson_apply(lat.h, out[r], src[r], kappa, p, prec)
            bq.bq_dd_unpack(lat.h, out[r], recv[r], -kappa, p, prec)
        torch.cuda.synchronize()
        assert relmax(R.export_field(out, prec, p), bqo.hop_restricted(U, psi, kappa, p)) < TOL[prec]
    finally:
        R.close()


@pytest.mark.parametrize("grid", [(2, 1, 1, 2), (1, 2, 2, 1)])
def test_dd_solve(bq, grid):
    """fp64 even-odd BiCGStab over virtual ranks: the solution, assembled from the ranks' blocks, judged with the oracle's
    operator on the global lattice; and it agrees with the single-GPU solve of the same system."""
    L, kappa = (8, 8, 8, 16), 0.1215
    U = inputs.gauge(L, 1207, 0.5)
    b = inputs.spinor(L, 1208)
    R = Ranks(bq, L, grid, U)
    try:
        bs = [dd.local_block(b, L, grid, dd.coords_of(r, grid)) for r in range(R.n)]
        xs = [np.zeros_like(v) for v in bs]
        info = bq.bq_dd_solve(R.handles(), bs, xs, kappa, 1e-10)
    finally:
        R.close()
    x = dd.assemble(xs, L, grid)
    res = np.linalg.norm(b - bqo.dirac_apply(U, x, kappa)) / np.linalg.norm(b)
    print(f"dd solve grid {grid}: {info.inner_iters} iterations, Schur residual {info.true_rel_residual:.2e}, oracle residual {res:.2e}")
    assert info.status == 0 and res <= 1e-10
    x1 = np.zeros_like(b)
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        info1 = bq.bq_solve(lat.h, b, x1, kappa, 1e-10, bq.bq_solve_opts(inner_prec=bq.BQ_FP64))
    assert np.linalg.norm(x - x1) / np.linalg.norm(x1) < 1e-8
    assert abs(info.inner_iters - info1.inner_iters) <= 2


def test_dd_errors(bq):
    L, grid = (8, 4, 4, 8), (2, 1, 1, 1)
    U = inputs.gauge(L, 1209, 0.3)
    with pytest.raises(bq.BqError):
        bq.bq_lattice_create_sub(4, 4, 4, 8, (2, 1, 1, 1), (2, 0, 0, 0))       # coordinate outside the grid
    R = Ranks(bq, L, grid, U)
    try:
        b = dd.local_block(inputs.spinor(L, 1210), L, grid, (0, 0, 0, 0))
        with pytest.raises(bq.BqError):                                          # a sub-lattice does not solve on its own
            bq.bq_solve(R.lats[0].h, b, np.zeros_like(b), 0.12, 1e-10)
        with pytest.raises(bq.BqError):                                          # clover is not built on sub-lattices
            bq.bq_clover_apply(R.lats[0].h, 1.0, 0.12, None, None, bq.BQ_FULL, 0, bq.BQ_FP64)
        # on a handle with a partitioned direction only bq_wilson_apply (the documented interior hop) runs; the composite
        # operators would return an interior-only result and refuse instead
        lat0 = R.lats[0]
        fo, fe, ft = lat0.field(bq.BQ_FP32, bq.BQ_ODD), lat0.field(bq.BQ_FP32, bq.BQ_EVEN), lat0.field(bq.BQ_FP32, bq.BQ_EVEN)
        full_in, full_out = lat0.field(bq.BQ_FP32, bq.BQ_FULL), lat0.field(bq.BQ_FP32, bq.BQ_FULL)
        bq.bq_wilson_apply(lat0.h, fe, fo, 0.12, bq.BQ_EVEN, bq.BQ_FP32)
        bq.bq_wilson_apply(lat0.h, full_out, full_in, 0.12, bq.BQ_FULL, bq.BQ_FP32)
        for call in (lambda: bq.bq_dirac_apply(lat0.h, full_out, full_in, 0.12, 0.0, bq.BQ_FP32),
                     lambda: bq.bq_schur_apply(lat0.h, fe, ft, fo, 0.12, 0.0, bq.BQ_FP32),
                     lambda: bq.bq_dirac_apply_mode(lat0.h, full_out, full_in, None, 0.12, 0.0, bq.BQ_MODE_DDAG, bq.BQ_FP32),
                     lambda: bq.bq_schur_apply_mode(lat0.h, fe, ft, fo, None, 0.12, 0.0, bq.BQ_MODE_D, bq.BQ_FP32),
                     lambda: bq.bq_wilson_apply_multi(lat0.h, fe, fo, 1, 0.12, bq.BQ_EVEN, bq.BQ_FP32),
                     lambda: bq.bq_schur_apply_multi(lat0.h, fe, ft, fo, 1, 0.12, 0.0, bq.BQ_FP32)):
            with pytest.raises(bq.BqError) as e:
                call()
            assert e.value.status == bq.BQ_EINVAL and "interior" in str(e.value)
        with pytest.raises(bq.BqError):                                          # one handle for a two-rank grid
            src = R.lats[0].field(bq.BQ_FP32, bq.BQ_ODD)
            bq.bq_dd_wilson_apply([R.lats[0].h], [R.lats[0].field(bq.BQ_FP32)], [src], 0.12, 0, bq.BQ_FP32)
    finally:
        R.close()


@pytest.mark.parametrize("prec", [0, 1])
def test_distributed_hop_single_rank(bq, prec):
    """dd.DistributedHop.apply — the call a process per GPU makes — executed on the one GPU with a 1 x 1 x 1 x 1 grid: no face
    leaves the rank, so no process group is needed, but the whole sequence runs: pack on the side stream, the interior hop on
    the current (non-default) stream, the wait, unpack.  The result is the oracle's hop on the global lattice."""
    import torch
    L, grid, kappa = (8, 4, 4, 8), (1, 1, 1, 1), 0.125
    U = inputs.gauge(L, 1211, 0.5)
    psi = inputs.spinor(L, 1212)
    R = Ranks(bq, L, grid, U, GENERAL_BC)
    try:
        hop = dd.DistributedHop(bq, R.lats[0], 0, grid, prec)
        assert all(b is None for b in hop.send + hop.recv)
        work = torch.cuda.Stream()
        for p in (0, 1):
            src = R.import_field(psi, prec, 1 - p)[0]
            out = R.lats[0].field(prec, p)
            torch.cuda.synchronize()
            with torch.cuda.stream(work):
                hop.apply(out, src, kappa, p)
            work.synchronize()
            ref = bqo.hop_restricted(U, psi, kappa, p, bc=GENERAL_BC)
            assert relmax(R.export_field([out], prec, p), ref) < TOL[prec]
    finally:
        R.close()
