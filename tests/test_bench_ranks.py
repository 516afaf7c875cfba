"""The N>1 path of bench.py on the CPU: two gloo ranks, max-over-ranks timing and whole-job throughput
(one process per GPU in the real run; rows are independent, so ranks are replicas with no data-path collective)."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, {root!r})
    import torch.distributed as dist
    import bench
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo")
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")      # rank 1 is the slow one
    v = bench.job_throughput(1000.0, 4, ms, world)
    dist.barrier()
    if rank == 0:
        print("RESULT", ms, v)
    dist.destroy_process_group()
""")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_ranks_max_time_and_sum_of_work(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=180) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    line = [ln for ln in outs[0][0].splitlines() if ln.startswith("RESULT")][0].split()
    ms, v = float(line[1]), float(line[2])
    assert ms == 15.0                                   # the slowest rank's time
    assert abs(v - 2 * 1000.0 * 4 / 15e-3) < 1e-6       # both ranks' work over that time


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.job_throughput(10.0, 2, 4.0, 1) == 5000.0
