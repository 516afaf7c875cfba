"""The N>1 path of bench.py on the CPU: two (and three) gloo ranks run the sharded build's host logic on real data —
per-cell hit counts from the oracle's count pass, the library's partitioner (pm_partition_cells, host only), one shard
per rank (built by the oracle here: there is no GPU), the all-gather of the per-rank nnz, the row-pointer offsets — and
rank 0 checks that the shards concatenate to the whole matrix.  SURVEY.md sec. 8(e); PAPER.md:L260 (independent elements)."""
import os
import socket
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, {root!r})
    import numpy as np
    import torch.distributed as dist
    import bench
    from oracle.pm_oracle import Oracle
    from paper_1508_07441_b200 import api, inputs as I
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo")
    o = Oracle(); o.set_threads(1)
    wl = I.small_coupled(N=5, jmax=1, orders=(3, 2, 5), Nq=6)
    # count pass, split evenly; every rank ends up with all hit counts
    lo, hi = wl.n_cells * rank // world, wl.n_cells * (rank + 1) // world
    hp, _ = o.hit_cells(wl, lo, hi)
    parts = [None] * world
    dist.all_gather_object(parts, np.diff(hp).astype(np.int32))
    hits = np.concatenate(parts)
    cuts, cell_cost = bench.shard_cuts(api, hits, world)          # pm_partition_cells: the same on every rank
    cb, ce = int(cuts[rank]), int(cuts[rank + 1])
    rp, ci, v = o.build_csr(wl, cb, ce)                            # this rank's shard (block-local row pointers)
    nnz_r = bench.gather_counts(int(rp[-1]), world, device="cpu")  # the one exchange
    off, total = bench.shard_offsets(nnz_r)
    rp_global = rp + off[rank]
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")      # the last rank is the slow one
    out = [None] * world
    dist.gather_object((cuts.tolist(), rp_global, ci, v), out if rank == 0 else None, dst=0)
    if rank == 0:
        rpo, cio, vo = o.build_csr(wl)
        assert all(p[0] == out[0][0] for p in out), "ranks disagree on the cuts"
        rows = np.concatenate([p[1][:-1] if k < world - 1 else p[1] for k, p in enumerate(out)])
        assert np.array_equal(rows, rpo) and total == rpo[-1]
        assert np.array_equal(np.concatenate([p[2] for p in out]), cio)
        assert np.array_equal(np.concatenate([p[3] for p in out]), vo)
        w = hits + cell_cost
        loads = [w[cuts[r]:cuts[r + 1]].sum() for r in range(world)]
        assert max(loads) <= w.sum() / world + w.max()
        print("RESULT", ms, bench.job_throughput(float(total), 4, ms), total)
    dist.barrier()
    dist.destroy_process_group()
""")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_build_host_logic_over_gloo(tmp_path, world):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE=str(world), LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port),
                   OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=600) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    line = [ln for ln in outs[0][0].splitlines() if ln.startswith("RESULT")][0].split()
    ms, v, total = float(line[1]), float(line[2]), float(line[3])
    assert ms == 10.0 + 5.0 * (world - 1)               # the slowest rank's time
    assert abs(v - total * 4 / (ms * 1e-3)) < 1e-6 * v  # ONE matrix over that time (strong scaling), not world copies of it


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.job_throughput(10.0, 2, 4.0) == 5000.0
    assert bench.gather_counts(7, 1) == [7]
    assert bench.shard_offsets([5, 0, 7]) == ([0, 5, 5], 12)
