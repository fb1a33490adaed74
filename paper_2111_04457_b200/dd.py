"""Domain decomposition helpers (opt-in; include/bq.h "Domain decomposition").

No field arithmetic lives here (every operation on a vector is a kernel of libbq.so; DistributedSolver advances only the
four complex scalars of the BiCGStab recurrence from all-reduced sums): rank <-> coordinates, cutting a global canonical array into the ranks' local
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


def sum_over_ranks(values, group=None, on_host=True):
    """The all-reduce of one reduction point of the distributed solver: the packed list of this rank's partial sums -> their
    sums over all ranks, as floats (a CPU tensor for gloo, a device tensor for NCCL).  One collective per call."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device="cpu" if on_host else "cuda")
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, group=group)
    return t.tolist()


class DistributedHop:
    """One process per GPU: out = -kappa H_{p,1-p} in on this rank's sub-lattice, halo exchange through torch.distributed.
    pack runs on a side stream and the interior hop on the current stream, enqueued BEFORE the host waits for any
    transfer (the communication is overlapped with the bulk); unpack follows both.
    host_staging=False: the face buffers travel as device tensors (NCCL over NVLink).  host_staging=True: they are copied
    to pinned host tensors on the side stream, exchanged there (the gloo backend moves CPU tensors only) and copied back —
    the form the GPU test runs with two processes sharing the one GPU.  UNMEASURED on multi-GPU hardware."""

    def __init__(self, bq, lat, rank, grid, prec, group=None, host_staging=False):
        import torch
        self.bq, self.lat, self.rank, self.grid, self.prec, self.group = bq, lat, rank, tuple(grid), prec, group
        self.host = bool(host_staging)
        self.side = torch.cuda.Stream()
        dt = torch.float64 if prec == bq.BQ_FP64 else torch.float32
        self.send, self.recv = [None] * 8, [None] * 8
        self.h_send, self.h_recv = [None] * 8, [None] * 8
        for mu in range(4):
            if self.grid[mu] > 1:
                n = bq.bq_dd_face_bytes(lat.h, mu, prec) // (8 if prec == bq.BQ_FP64 else 4)
                for s in range(2):
                    self.send[2 * mu + s] = torch.empty(n, dtype=dt, device="cuda")
                    self.recv[2 * mu + s] = torch.empty(n, dtype=dt, device="cuda")
                    if self.host:
                        self.h_send[2 * mu + s] = torch.empty(n, dtype=dt).pin_memory()
                        self.h_recv[2 * mu + s] = torch.empty(n, dtype=dt).pin_memory()

    def apply(self, out, inp, kappa, parity, recon=0):
        import torch
        bq, cur = self.bq, torch.cuda.current_stream()
        self.side.wait_stream(cur)
        with torch.cuda.stream(self.side):
            bq.bq_dd_pack(self.lat.h, self.send, inp, parity, self.prec, recon, self.side)
            if self.host:
                for d, h in zip(self.send, self.h_send):
                    if d is not None:
                        h.copy_(d, non_blocking=True)
        bq.bq_wilson_apply(self.lat.h, out, inp, kappa, parity, self.prec, recon, cur)      # interior
        with torch.cuda.stream(self.side):
            if self.host:
                self.side.synchronize()                       # the packed faces are on the host
                exchange_faces(self.h_send, self.h_recv, self.rank, self.grid, self.group)
                for d, h in zip(self.recv, self.h_recv):
                    if d is not None:
                        d.copy_(h, non_blocking=True)
            else:
                exchange_faces(self.send, self.recv, self.rank, self.grid, self.group)
        cur.wait_stream(self.side)
        bq.bq_dd_unpack(self.lat.h, out, self.recv, -kappa, parity, self.prec, recon, cur)


class DistributedSolver:
    """One process per GPU: D x = b for the Wilson matrix (csw = 0) on the GLOBAL lattice, each rank holding its local block —
    the even-odd Schur system M^ x_e = b^_e, M^ = 1 - kappa^2 H_eo H_oe, solved by fp64 BiCGStab (reading O4, the recurrences
    of bq_dd_solve / solve.cu), then x_o = b_o + kappa H_oe x_e.  Every operator application is two DistributedHop.apply
    calls (halo exchange per hop); every vector operation is one of the library's fused BLAS-1 kernels on the rank's fields;
    every inner product is the rank's device reduction followed by ONE torch.distributed.all_reduce of the packed scalars of
    that reduction point (2, 3 and 3 doubles per iteration) — the only places where the ranks meet besides the faces.  The
    handful of complex scalars (rho, alpha, omega, beta) are advanced here on the host, identically on every rank, from the
    all-reduced sums.  UNMEASURED on multi-GPU hardware; tested with two processes sharing one GPU over gloo."""

    def __init__(self, bq, lat, rank, grid, group=None, host_staging=False):
        self.bq, self.lat, self.group, self.host = bq, lat, group, bool(host_staging)
        self.hop = DistributedHop(bq, lat, rank, grid, bq.BQ_FP64, group, host_staging)

    def _sum_over_ranks(self, values):
        return sum_over_ranks(values, self.group, on_host=self.host)

    def _schur(self, out, inp, tmp_o, tmp_e, kappa):
        """out = M^ inp = inp - (-kappa H_eo)(-kappa H_oe) inp."""
        bq = self.bq
        self.hop.apply(tmp_o, inp, kappa, bq.BQ_ODD)
        self.hop.apply(tmp_e, tmp_o, kappa, bq.BQ_EVEN)
        out.copy_(inp)
        bq.bq_blas_caxpy(self.lat.h, -1.0, tmp_e, out, bq.BQ_FP64)

    def solve(self, b_local, x_local, kappa, tol, max_iter=1000):
        """b_local: this rank's canonical complex128 block [lt, lz, ly, lx, 4, 3]; x_local: same shape, receives the solution
        (zero initial guess).  Returns {"iters", "schur_rel_residual", "converged"}."""
        import torch
        bq, lat = self.bq, self.lat
        P64, h = bq.BQ_FP64, lat.h
        fb = bq.bq_field_bytes(h, P64, bq.BQ_EVEN)
        bfull = lat.import_field(b_local, P64, bq.BQ_FULL)
        be, bo = bfull[:fb], bfull[fb:]
        new = lambda: lat.field(P64, bq.BQ_EVEN)
        bnorm2, = self._sum_over_ranks([bq.bq_blas_norm2(h, be, P64) + bq.bq_blas_norm2(h, bo, P64)])
        x, tmp_o, tmp_e, v, s, t, ptmp = new(), new(), new(), new(), new(), new(), new()
        # b^_e = b_e + kappa H_eo b_o
        self.hop.apply(tmp_e, bo, kappa, bq.BQ_EVEN)
        bhat = be.clone()
        bq.bq_blas_caxpy(h, -1.0, tmp_e, bhat, P64)
        r = bhat.clone()
        rhat, p = r.clone(), r.clone()
        r2, = self._sum_over_ranks([bq.bq_blas_norm2(h, r, P64)])
        rho = complex(r2, 0.0)
        target2 = tol * tol * bnorm2
        iters, converged = 0, r2 <= target2
        while not converged and iters < max_iter:
            self._schur(v, p, tmp_o, tmp_e, kappa)
            d = bq.bq_blas_cdot(h, rhat, v, P64)
            re, im = self._sum_over_ranks([d.real, d.imag])
            rv = complex(re, im)
            if rv == 0 or rho == 0:
                break                                               # breakdown
            alpha = rho / rv
            s.copy_(r)
            bq.bq_blas_caxpy(h, -alpha, v, s, P64)
            self._schur(t, s, tmp_o, tmp_e, kappa)
            d = bq.bq_blas_cdot(h, t, s, P64)
            re, im, tt = self._sum_over_ranks([d.real, d.imag, bq.bq_blas_norm2(h, t, P64)])
            if tt == 0:
                break
            omega = complex(re, im) / tt
            lr2, lrr = bq.bq_blas_bicg_update(h, alpha, omega, p, s, t, rhat, x, r, P64)     # x += alpha p + omega s; r = s - omega t
            r2, re, im = self._sum_over_ranks([lr2, lrr.real, lrr.imag])
            iters += 1
            if r2 <= target2:
                converged = True
                break
            rho_new = complex(re, im)
            if omega == 0:
                break
            beta = (rho_new / rho) * (alpha / omega)
            rho = rho_new
            bq.bq_blas_caxpy(h, -omega, v, p, P64)                   # p = r + beta (p - omega v)
            ptmp.copy_(r)
            bq.bq_blas_caxpy(h, beta, p, ptmp, P64)
            p, ptmp = ptmp, p
        # the residual of the Schur system, recomputed with the operator
        self._schur(t, x, tmp_o, tmp_e, kappa)
        bq.bq_blas_caxpy(h, -1.0, t, bhat, P64)
        res2, = self._sum_over_ranks([bq.bq_blas_norm2(h, bhat, P64)])
        # x_o = b_o + kappa H_oe x_e
        self.hop.apply(tmp_o, x, kappa, bq.BQ_ODD)
        xo = bo.clone()
        bq.bq_blas_caxpy(h, -1.0, tmp_o, xo, P64)
        torch.cuda.synchronize()
        xfull = torch.cat([x, xo])
        x_local[...] = lat.export_field(xfull, P64, bq.BQ_FULL)
        rel = (res2 / bnorm2) ** 0.5 if bnorm2 > 0 else 0.0
        return {"iters": iters, "schur_rel_residual": rel, "converged": bool(rel <= tol)}
