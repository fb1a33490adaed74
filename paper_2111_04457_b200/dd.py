"""Domain decomposition helpers (opt-in; include/bq.h "Domain decomposition").

No arithmetic of the method lives here: rank <-> coordinates, cutting a global canonical array into the ranks' local
blocks (array slicing), the schedule of the halo exchange (who sends which face to whom), and — for one process per
GPU — the transport of the face buffers between bq_dd_pack and bq_dd_unpack through torch.distributed point-to-point
calls (NCCL over NVLink on GPUs; the same schedule runs on the gloo backend with CPU tensors, which is how it is tested
here).  The multi-process path is UNMEASURED on hardware: no multi-GPU node was available to this build.
"""
from __future__ import annotations

import numpy as np


def coords_of(rank, grid):
    """Rank number -> grid coordinates, x fastest (the convention of bq_lattice_create_sub)."""
    c = []
    for g in grid:
        c.append(rank % g)
        rank //= g
    return tuple(c)


def rank_of(coords, grid):
    r = 0
    for c, g in zip(reversed(coords), reversed(grid)):
        r = r * g + c
    return r


def local_extents(L, grid):
    assert all(l % g == 0 and (l // g) % 2 == 0 for l, g in zip(L, grid)), "every local extent must be even"
    return tuple(l // g for l, g in zip(L, grid))


def local_block(field, L, grid, coords):
    """The local block of a global canonical array [Lt, Lz, Ly, Lx, ...] (a copy, C-contiguous)."""
    lx, ly, lz, lt = local_extents(L, grid)
    cx, cy, cz, ct = coords
    return np.ascontiguousarray(field[ct * lt:(ct + 1) * lt, cz * lz:(cz + 1) * lz, cy * ly:(cy + 1) * ly, cx * lx:(cx + 1) * lx])


def assemble(blocks, L, grid):
    """Inverse of local_block over all ranks: blocks[rank] -> global array."""
    lx, ly, lz, lt = local_extents(L, grid)
    out = np.zeros((L[3], L[2], L[1], L[0]) + blocks[0].shape[4:], dtype=blocks[0].dtype)
    for r, b in enumerate(blocks):
        cx, cy, cz, ct = coords_of(r, grid)
        out[ct * lt:(ct + 1) * lt, cz * lz:(cz + 1) * lz, cy * ly:(cy + 1) * ly, cx * lx:(cx + 1) * lx] = b
    return out


def face_schedule(rank, grid):
    """The halo exchange of one hop as seen from `rank`: a list of transfers
        (mu, send_side, dest_rank, recv_side, source_rank)
    meaning: the face packed as send[2*mu + send_side] goes to dest_rank, and recv[2*mu + recv_side] is filled by what
    source_rank packed as ITS send[2*mu + send_side].  Side 0 (slice x_mu = 0) travels DOWN and lands in the lower rank's
    recv side 1 (its slice x_mu = l_mu - 1); side 1 travels UP and lands in the upper rank's recv side 0.  Unpartitioned
    directions do not appear.  With two ranks in a direction the lower and the upper neighbour are the same rank: both
    transfers still happen (two different faces)."""
    c = coords_of(rank, grid)
    out = []
    for mu in range(4):
        if grid[mu] == 1:
            continue
        lo, hi = list(c), list(c)
        lo[mu] = (c[mu] - 1) % grid[mu]
        hi[mu] = (c[mu] + 1) % grid[mu]
        below, above = rank_of(lo, grid), rank_of(hi, grid)
        out.append((mu, 0, below, 1, above))     # our side 0 -> below; our recv side 1 <- above's side 0
        out.append((mu, 1, above, 0, below))     # our side 1 -> above; our recv side 0 <- below's side 1
    return out


def exchange_faces(send, recv, rank, grid, group=None):
    """Move the packed faces of one hop: send / recv are lists of 8 tensors (index 2*mu + side; None where unpartitioned),
    on the device for NCCL or on the CPU for gloo.  Non-blocking point-to-point operations, one batch per hop; returns after
    every transfer has completed.  The tag encodes (mu, send_side) so that the two faces exchanged by a pair of ranks in a
    direction of extent two cannot be confused."""
    import torch.distributed as dist
    ops = []
    for mu, sside, dest, rside, src in face_schedule(rank, grid):
        ops.append(dist.P2POp(dist.isend, send[2 * mu + sside], dest, group=group, tag=2 * mu + sside))
        ops.append(dist.P2POp(dist.irecv, recv[2 * mu + rside], src, group=group, tag=2 * mu + sside))
    if not ops:
        return
    for req in dist.batch_isend_irecv(ops):
        req.wait()


class DistributedHop:
    """One process per GPU: out = -kappa H_{p,1-p} in on this rank's sub-lattice, halo exchange through torch.distributed.
    pack and the transfers run on a side stream while the interior hop runs on the current stream (the
    communication is overlapped with the bulk); unpack follows both.  UNMEASURED on hardware."""

    def __init__(self, bq, lat, rank, grid, prec, group=None):
        import torch
        self.bq, self.lat, self.rank, self.grid, self.prec, self.group = bq, lat, rank, tuple(grid), prec, group
        self.side = torch.cuda.Stream()
        dt = torch.float64 if prec == bq.BQ_FP64 else torch.float32
        self.send, self.recv = [None] * 8, [None] * 8
        for mu in range(4):
            if self.grid[mu] > 1:
                n = bq.bq_dd_face_bytes(lat.h, mu, prec) // (8 if prec == bq.BQ_FP64 else 4)
                for s in range(2):
                    self.send[2 * mu + s] = torch.empty(n, dtype=dt, device="cuda")
                    self.recv[2 * mu + s] = torch.empty(n, dtype=dt, device="cuda")

    def apply(self, out, inp, kappa, parity, recon=0):
        import torch
        bq, cur = self.bq, torch.cuda.current_stream()
        self.side.wait_stream(cur)
        with torch.cuda.stream(self.side):
            bq.bq_dd_pack(self.lat.h, self.send, inp, parity, self.prec, recon, self.side)
            exchange_faces(self.send, self.recv, self.rank, self.grid, self.group)
        bq.bq_wilson_apply(self.lat.h, out, inp, kappa, parity, self.prec, recon, cur)      # interior
        cur.wait_stream(self.side)
        bq.bq_dd_unpack(self.lat.h, out, self.recv, -kappa, parity, self.prec, recon, cur)
