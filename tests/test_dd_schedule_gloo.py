"""The halo-exchange schedule of the opt-in domain decomposition (paper_2111_04457_b200/dd.py) on the CPU: pure-Python
consistency of face_schedule over whole grids, and a world_size-2 gloo run of exchange_faces with CPU tensors that carry
their origin — every receive buffer must end up holding exactly the face its neighbour packed for it."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_2111_04457_b200 import dd

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("grid", [(2, 1, 1, 2), (1, 1, 1, 2), (2, 2, 2, 2), (3, 1, 2, 4), (1, 1, 1, 1)])
def test_schedule_is_consistent(grid):
    n = int(np.prod(grid))
    for r in range(n):
        assert dd.rank_of(dd.coords_of(r, grid), grid) == r
    sends, recvs = set(), set()
    for r in range(n):
        sched = dd.face_schedule(r, grid)
        assert len(sched) == 2 * sum(g > 1 for g in grid)
        for mu, sside, dest, rside, src in sched:
            assert rside == 1 - sside
            cd, cs, c = dd.coords_of(dest, grid), dd.coords_of(src, grid), dd.coords_of(r, grid)
            step = -1 if sside == 0 else 1                    # side 0 travels down, side 1 up
            assert cd[mu] == (c[mu] + step) % grid[mu] and cs[mu] == (c[mu] - step) % grid[mu]
            assert all(cd[nu] == c[nu] == cs[nu] for nu in range(4) if nu != mu)
            sends.add((r, dest, mu, sside))
            recvs.add((src, r, mu, sside))
    assert sends == recvs                                     # every send is somebody's receive, and the other way round


def test_local_blocks_tile_the_lattice():
    L, grid = (8, 4, 12, 8), (2, 1, 3, 2)
    f = np.arange(np.prod(L) * 2, dtype=np.float64).reshape(L[3], L[2], L[1], L[0], 2)
    blocks = [dd.local_block(f, L, grid, dd.coords_of(r, grid)) for r in range(int(np.prod(grid)))]
    assert all(b.shape[:4] == (4, 4, 4, 4) for b in blocks)
    assert np.array_equal(dd.assemble(blocks, L, grid), f)


WORKER = r"""
import os, sys
import torch, torch.distributed as dist
sys.path.insert(0, os.environ["BQ_ROOT"])
from paper_2111_04457_b200 import dd
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
rank, grid = dist.get_rank(), (1, 1, 1, 2)
n = 24
# a face packed by rank r for (mu, side) carries 1000 r + 10 mu + side
send = [None] * 8
recv = [None] * 8
for mu in range(4):
    if grid[mu] > 1:
        for side in range(2):
            send[2 * mu + side] = torch.full((n,), float(1000 * rank + 10 * mu + side))
            recv[2 * mu + side] = torch.full((n,), -1.0)
for it in range(3):                                           # the same buffers hop after hop
    dd.exchange_faces(send, recv, rank, grid)
    for mu, sside, dest, rside, src in dd.face_schedule(rank, grid):
        want = float(1000 * src + 10 * mu + sside)
        assert torch.all(recv[2 * mu + rside] == want), (rank, mu, rside, recv[2 * mu + rside][0].item(), want)
# the packed scalars of one reduction point of dd.DistributedSolver: one all-reduce, identical sums on every rank
got = dd.sum_over_ranks([1.5 + rank, -2.0 * rank, 0.25], on_host=True)
assert got == [1.5 + 2.5, -2.0, 0.5], got
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_exchange_faces_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), BQ_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=120)[0] for p in procs]
    for rank, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"ok {rank}" in o, o
