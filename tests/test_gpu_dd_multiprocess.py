"""The process-per-GPU half of the opt-in domain decomposition ("parallelized with MPI", PAPER.md:95
halo exchange overlapped with the bulk), EXECUTED: two processes, one rank each, sharing the one GPU of the test box, the faces
travelling between them through the gloo backend (pinned host staging; on a multi-GPU node the same code moves device buffers with
NCCL).  Each process runs dd.DistributedHop.apply — pack on a side stream, interior hop on the current stream, exchange, unpack —
and dd.DistributedSolver.solve, whose inner products are all-reduced over the ranks.  The parent assembles the ranks' blocks and
judges them with the ORACLE on the global lattice.  No kernel of one rank waits for a kernel of the other: the processes meet only
on the host, between kernels."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from oracle import bqo
from paper_2111_04457_b200 import dd, inputs
from tests.conftest import relmax

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
import numpy as np
import torch, torch.distributed as dist
sys.path.insert(0, os.environ["BQ_ROOT"])
from paper_2111_04457_b200 import bq, dd
work = os.environ["BQ_WORK"]
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
torch.cuda.set_device(0)
dist.init_process_group("gloo", rank=rank, world_size=world)
meta = np.load(os.path.join(work, "meta.npy"))
L, grid, kappa = tuple(int(v) for v in meta[:4]), tuple(int(v) for v in meta[4:8]), 0.125
bc = np.load(os.path.join(work, "bc.npy"))
U = np.load(os.path.join(work, "U.npy")); psi = np.load(os.path.join(work, "psi.npy")); b = np.load(os.path.join(work, "b.npy"))
coords = dd.coords_of(rank, grid)
l = dd.local_extents(L, grid)
with bq.Lattice(l, bc, grid=grid, coords=coords) as lat:
    bq.bq_gauge_load(lat.h, dd.local_block(U, L, grid, coords))
    psi_l = dd.local_block(psi, L, grid, coords)
    for prec in (bq.BQ_FP64, bq.BQ_FP32):
        hop = dd.DistributedHop(bq, lat, rank, grid, prec, host_staging=True)
        for p in (0, 1):
            src = lat.import_field(psi_l, prec, 1 - p)
            out = lat.field(prec, p)
            for rep in range(2):                      # the same buffers hop after hop
                hop.apply(out, src, kappa, p, recon=prec)    # 18-real in fp64, 12-real in fp32
            torch.cuda.synchronize()
            np.save(os.path.join(work, f"hop_{prec}_{p}_{rank}.npy"), lat.export_field(out, prec, p))
    solver = dd.DistributedSolver(bq, lat, rank, grid, host_staging=True)
    b_l = dd.local_block(b, L, grid, coords)
    x_l = np.zeros_like(b_l)
    info = solver.solve(b_l, x_l, 0.1215, 1e-10)
    np.save(os.path.join(work, f"x_{rank}.npy"), x_l)
    print("info", rank, info["iters"], info["schur_rel_residual"], info["converged"])
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_two_processes_one_gpu_hop_and_solve(tmp_path):
    L, grid = (8, 8, 8, 16), (1, 1, 1, 2)
    bc = np.exp(1j * np.array([0.4, -1.3, 2.0, 0.9]))
    U = inputs.gauge(L, 1301, 0.5)
    psi = inputs.spinor(L, 1302)
    b = inputs.spinor(L, 1303)
    np.save(tmp_path / "meta.npy", np.array(L + grid))
    np.save(tmp_path / "bc.npy", bc)
    np.save(tmp_path / "U.npy", U); np.save(tmp_path / "psi.npy", psi); np.save(tmp_path / "b.npy", b)
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), BQ_ROOT=ROOT,
                   BQ_WORK=str(tmp_path))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    outs = []
    try:
        for p in procs:
            outs.append(p.communicate(timeout=420)[0])
    finally:
        for p in procs:
            if p.poll() is None:
                p.kill()
    for rank, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"ok {rank}" in o, o
    # the hop, every site of the global lattice, both parities, general boundary phases
    for prec, tol in ((0, 1e-12), (1, 1e-5)):
        for p in (0, 1):
            got = dd.assemble([np.load(tmp_path / f"hop_{prec}_{p}_{r}.npy") for r in range(2)], L, grid)
            assert relmax(got, bqo.hop_restricted(U, psi, 0.125, p, bc=bc)) < tol, (prec, p)
    # the solve: residual recomputed with the oracle's operator on the global lattice
    x = dd.assemble([np.load(tmp_path / f"x_{r}.npy") for r in range(2)], L, grid)
    res = np.linalg.norm(b - bqo.dirac_apply(U, x, 0.1215, bc=bc)) / np.linalg.norm(b)
    print("two-process solve:", [ln for o in outs for ln in o.splitlines() if ln.startswith("info")], "oracle residual", res)
    assert res <= 1e-10
    # both ranks went through the same iteration (the all-reduced scalars are identical on every rank)
    its = [[ln.split()[2] for ln in o.splitlines() if ln.startswith("info")][0] for o in outs]
    assert its[0] == its[1]
