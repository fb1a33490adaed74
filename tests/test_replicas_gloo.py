"""N > 1 path on CPU: two gloo ranks run the replica plumbing bench.py uses (barrier, MAX over ranks of the per-rank
time, whole-job aggregate = world * units / slowest time).  DESIGN.md §7: replicas only, no data-path collective."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, {root!r})
    from paper_2111_04457_b200 import replicas
    rank, local_rank, world = replicas.env()
    assert replicas.init("gloo") == 2 and world == 2
    replicas.barrier()
    seconds = 0.5 if rank == 0 else 2.0                 # rank 1 is the slow replica
    mx = replicas.max_over_ranks(seconds)
    rate = replicas.whole_job_rate(1000.0, seconds)      # each rank processed 1000 units
    replicas.finish()
    print(json.dumps({{"rank": rank, "max": mx, "rate": rate}}))
""")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_gloo_replicas_agree_on_max_time_and_aggregate(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err
        outs.append(out.strip().splitlines()[-1])
    import json
    res = sorted((json.loads(o) for o in outs), key=lambda r: r["rank"])
    for r in res:
        assert r["max"] == 2.0                           # both ranks see the slowest replica's time
        assert r["rate"] == 2 * 1000.0 / 2.0             # whole-job aggregate over both replicas


def test_single_process_is_identity():
    from paper_2111_04457_b200 import replicas
    assert replicas.env()[2] == 1 or "WORLD_SIZE" in os.environ
    assert replicas.max_over_ranks(1.25) == 1.25
    assert replicas.whole_job_rate(10.0, 2.0) == 5.0


def test_reference_arm_runs_on_rank0_only(tmp_path):
    """bench.py --impl reference under a 2-rank launch: rank 1 exits 0 without output or work."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
