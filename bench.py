#!/usr/bin/env python
"""bench.py — P-matrix build throughput on B200 (BASELINE.json metric: nonzeros/s, build time, % FP64 peak).

A "step" is one pass of the whole hot path over one lattice through pm_build: the pattern pass (map and sort every
quadrature node, scan, row pointers) and the fill kernel, which writes the column index and the value of every nonzero; the default workload is BASELINE.json configs[4] (the largest lattice; its CSR fits HBM, one block).
`value` times the device-resident path with CUDA events; `e2e` times pm_build_host (host buffers, D2H copies
inside the timed region); `roofline` is for the dominant kernel (the fill); `cpu_baseline` times the oracle on
a bounded sample of source cells on the host cores (single thread and OpenMP).  `lattices` repeats the device-timed
build on all five BASELINE lattices (north_star: "throughput is reported at 1 GPU on the five synthetic lattices").
`--impl reference` times the oracle alone.  With N > 1 ranks ONE lattice is split over the ranks by contiguous source-cell
ranges balanced by hit count (strong scaling); the only exchange is an all-gather of the per-rank nnz.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1508_07441_b200 import inputs  # noqa: E402

METRIC = "P-matrix nonzeros/sec (pattern + fill, FP64)"
UNIT = "nnz/s"
# FP64 ALU peak used for the roofline: SMs x 64 DFMA lanes x 2 flop x max SM clock
FP64_LANES_PER_SM = 64
# dram__bytes_read.sum + dram__bytes_write.sum of one fill launch, QUOTED from the committed `ncu --set full` capture
# named beside it (bench.py cannot run under the profiler); None where no capture exists.
FILL_DRAM_TRAFFIC = {"cfg4_3N_Jhalf+_jle3_26ch_150x150": (10.777e9 + 0.318e9, "profiles/r2_final.md (ncu --set full of this kernel, round 2; quoted, not measured in this run)")}


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return {"hbm_gbs": d.get("hbm_gbs", 6650.0), "sm_max_mhz": d.get("sm_max_mhz", 1965.0), "src": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "src": "fallback"}


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons every 50 ms during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.out = index, None, ""

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "50"], stdout=subprocess.PIPE, text=True)
            time.sleep(0.25)                        # let the first samples arrive before the timed region starts
        except Exception:
            self.proc = None
        return self

    def __exit__(self, *a):
        if self.proc is not None:
            time.sleep(0.1)
            self.proc.terminate()
            try:
                self.out = self.proc.communicate(timeout=5)[0]
            except Exception:
                self.out = ""

    def summary(self):
        sm, mx, pw, reasons = [], 0.0, [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.out.strip().splitlines():
            r = [c.strip() for c in line.split(",")]
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1])); pw.append(float(r[2]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "power_w_max": max(pw) if pw else None, "samples": len(sm)}


def max_over_ranks(x: float, world: int, device="cuda") -> float:
    """Max of a per-rank scalar over all ranks (device time of the slowest rank); identity for one rank."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_step: float, steps: int, total_ms: float) -> float:
    """Whole-job units per second: `units_per_step` is what ALL ranks together process per step (one lattice split over
    the ranks), `total_ms` the max over ranks of the time for `steps` steps."""
    return units_per_step * steps / (total_ms * 1e-3)


def gather_counts(x: int, world: int, device="cuda"):
    """All-gather of one int64 per rank (the per-shard nnz: the only exchange of the sharded build)."""
    if world <= 1:
        return [int(x)]
    import torch
    import torch.distributed as dist
    mine = torch.tensor([int(x)], dtype=torch.int64, device=device)
    out = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(out, mine)
    return [int(t.item()) for t in out]


def shard_offsets(nnz_per_rank):
    """Exclusive prefix of the per-rank nnz: what a rank adds to its block-local row pointers."""
    off, run = [], 0
    for n in nnz_per_rank:
        off.append(run); run += int(n)
    return off, run


def shard_cuts(api, hits, world):
    """Contiguous source-cell ranges balanced by hit count (pm_partition_cells; the same on every rank).  A cell's cost is
    its hit cells (row writes) plus a constant for its quadrature nodes; the constant comes from the fill's profile
    (node phases ~58 % of the warp time, per-target phases ~42 %)."""
    import numpy as _np
    cell_cost = 1.4 * float(_np.mean(hits)) if len(hits) else 0.0
    return api.pm_partition_cells(hits, world, cell_cost), cell_cost


def build_flops(lat_api, h):
    """Algorithmic FP64 flops of one build: pm_lattice_work x pm_pattern_counts."""
    per_node, per_seg, per_hit, _ = lat_api.pm_lattice_work(h)
    nodes, segs, hits = lat_api.pm_pattern_counts(h)
    return per_node * nodes + per_seg * segs + per_hit * hits, {"flop_per_node": per_node, "flop_per_segment": per_seg,
                                                                 "flop_per_hit_cell": per_hit, "nodes_on_grid": nodes,
                                                                 "segments": segs, "hit_cells": hits}


def oracle_sample(wl, seconds_target=10.0, threads=None, batch=None):
    """Times the oracle as it stands on evenly spaced batches of consecutive source cells of `wl` (bounded CPU work).
    po_build's OpenMP loop runs over the source cells of one call, so a call gets `batch` >= 4 x threads cells."""
    from oracle.pm_oracle import Oracle
    o = Oracle()
    if threads:
        o.set_threads(threads)
    nthr = o.threads()
    batch = batch or max(1, 4 * nthr)
    starts = np.unique(np.linspace(0, max(0, wl.n_cells - batch), 64).astype(int))
    t0 = time.perf_counter()
    nnz, cells = 0, 0
    for c0 in starts:
        c1 = min(wl.n_cells, int(c0) + batch)
        rp, _, _ = o.build_csr(wl, int(c0), c1)
        nnz += int(rp[-1]); cells += c1 - int(c0)
        if time.perf_counter() - t0 > seconds_target:
            break
    dt = time.perf_counter() - t0
    return {"value": nnz / dt, "unit": UNIT, "threads": nthr, "cells": cells, "nnz": nnz, "seconds": dt, "cells_per_call": batch}


def cpu_baseline(wl, seconds=10.0):
    """The oracle on the host cores: OpenMP over the source cells of a call (all threads) and one thread."""
    ncpu = os.cpu_count() or 1
    omp = oracle_sample(wl, seconds, threads=ncpu)
    one = oracle_sample(wl, max(3.0, seconds / 2), threads=1, batch=4)
    return {"value": omp["value"], "unit": UNIT, "cores": omp["threads"], "kind": "oracle",
            "single_thread": {"value": one["value"], "threads": 1, "cells": one["cells"], "seconds": round(one["seconds"], 2)},
            "openmp": {"value": omp["value"], "threads": omp["threads"], "cells": omp["cells"], "seconds": round(omp["seconds"], 2)},
            "sample": f"evenly spaced batches of {omp['cells_per_call']} consecutive source cells of {wl.name}: {omp['cells']} cells, "
                      f"{omp['nnz']} nnz in {omp['seconds']:.1f} s on {omp['threads']} OpenMP threads; single thread: {one['cells']} cells in {one['seconds']:.1f} s"}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    wl = inputs.config(args.config if args.config != "all" else 4)
    ncpu = os.cpu_count() or 1
    per_step = max(2.0, min(15.0, 100.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(wl, per_step, threads=ncpu)
    tot_nnz, tot_t, last = 0, 0.0, None
    for _ in range(args.steps):
        last = oracle_sample(wl, per_step, threads=ncpu)
        tot_nnz += last["nnz"]; tot_t += last["seconds"]
    one = oracle_sample(wl, 4.0, threads=1, batch=4)
    v = tot_nnz / tot_t
    info = {"value": v, "unit": UNIT, "cores": last["threads"], "kind": "oracle",
            "single_thread": {"value": one["value"], "threads": 1}, "openmp": {"value": v, "threads": last["threads"]},
            "sample": f"per step: evenly spaced batches of {last['cells_per_call']} consecutive source cells of {wl.name} for {per_step:.0f} s "
                      f"({last['cells']} cells in the last step) on {last['threads']} OpenMP threads"}
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
                      "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
                      "data": "synthetic", "config": {"workload": wl.name, "M": wl.M, "sampled": True},
                      "cpu_baseline": info,
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def timed_builds(api, torch, lat, wl, cb, ce, rowptr, colidx, vals, flush, steps, warmup, world, barrier, st, sampler=None):
    """`steps` timed pm_build calls on source cells [cb, ce) (CUDA events on the launching stream, L2 flushed in between).
    Returns (per-step ms, per-step fill-kernel ms, nnz of the range, launches in the timed region)."""
    nnz = 0
    for _ in range(max(warmup, 3)):
        nnz = api.pm_build(lat.h, cb, ce, rowptr, colidx, vals)
    barrier()
    l0 = api.pm_launch_count()
    step_ms, fill_ms = [], []
    ctx = sampler if sampler is not None else _Null()
    with ctx:
        for _ in range(steps):
            flush.zero_()                                     # L2 flush between timed iterations (untimed)
            e0, e1 = (torch.cuda.Event(enable_timing=True) for _ in range(2))
            barrier()
            e0.record(st)
            n_r = api.pm_build(lat.h, cb, ce, rowptr, colidx, vals)
            if world > 1:                                     # the one exchange of the sharded build: per-rank nnz -> row-pointer offsets
                off, _ = shard_offsets(gather_counts(n_r, world))
                api.pm_rowptr_offset(rowptr, off[int(os.environ.get("RANK", "0"))])
            e1.record(st)
            torch.cuda.synchronize()
            step_ms.append(e0.elapsed_time(e1))
            fill_ms.append(api.pm_last_fill_ms(lat.h) if ce > cb else 0.0)     # CUDA events around the fill kernel, on its stream
        barrier()
    return step_ms, fill_ms, nnz, api.pm_launch_count() - l0


class _Null:
    def __enter__(self):
        return self

    def __exit__(self, *a):
        return False


def fill_roofline(api, lat, wl, nnz, fill_ms, pk, n_sm, dfma):
    """Both roofs of the fill kernel, the binding one first.  HBM: algorithmic bytes = 12 B per nonzero
    written once; the 8-byte chunk words the kernel reads (one per run of at most four nodes) are listed
    separately."""
    peak_tf = n_sm * FP64_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 * 1e-12
    flops, work = build_flops(api, lat.h)
    fill_avg = float(np.mean(fill_ms)) * 1e-3
    achieved_tf = flops / fill_avg * 1e-12
    alg_bytes = 12.0 * nnz
    key_bytes = 8.0 * api.pm_pattern_chunks(lat.h)
    achieved_gbs = alg_bytes / fill_avg * 1e-9
    t_alu, t_hbm = flops / (peak_tf * 1e12), alg_bytes / (pk["hbm_gbs"] * 1e9)
    alu = {"achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved_tf / peak_tf,
           "peak_source": f"{n_sm} SM x {FP64_LANES_PER_SM} DFMA lanes x 2 x {pk['sm_max_mhz']:.0f} MHz ({pk['src']} clock)"
                          + (f"; DFMA microbenchmark on this box: {dfma:.1f} TFLOP/s" if dfma else "")}
    hbm = {"achieved": achieved_gbs, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": achieved_gbs / pk["hbm_gbs"],
           "peak_source": f"copy bandwidth, MEASURED_PEAKS.json ({pk['src']})"}
    bound = "hbm" if t_hbm >= t_alu else "alu"
    traffic, traffic_src = FILL_DRAM_TRAFFIC.get(wl.name, (None, None))
    return {"bound": bound, "kernel": "k_fill_warp (values + column indices)", **(hbm if bound == "hbm" else alu),
            "traffic": traffic, "traffic_source": traffic_src, "algorithmic_bytes": alg_bytes, "chunk_word_bytes_read": key_bytes,
            "flops_per_launch": flops, "flop_per_byte": flops / alg_bytes, "ridge_flop_per_byte": peak_tf * 1e3 / pk["hbm_gbs"],
            "min_ms": {"alu": t_alu * 1e3, "hbm": t_hbm * 1e3}, "alu": alu, "hbm": hbm, "work": work, "fill_ms": fill_avg * 1e3}


def jpi_sweep(api, torch, lat, wl, flush, st):
    """SURVEY sec. 8(f) rank 3 / PAPER.md Table 1 (L396-404: '62 spin-orbital channels and all states ... up to J_max = 17/2'):
    every J^pi <= 17/2 (pair j <= 3) on the grid of `wl`, each attached to the base lattice and built with pm_build_reuse into
    one pair of buffers sized for the largest set; the geometric pattern (map + sort) is computed once, before the sweep."""
    rp = torch.empty(wl.n_cells * 64 + 1, dtype=torch.int64, device="cuda")
    e0, e1 = (torch.cuda.Event(enable_timing=True) for _ in range(2))
    e0.record(st)
    nnz0 = api.pm_pattern(lat.h, 0, wl.n_cells, rp, None)                # the one node map + sort of the sweep
    e1.record(st); torch.cuda.synchronize()
    pattern_ms = e0.elapsed_time(e1)
    hits = nnz0 // int(api.pm_lattice_coupling(lat.h, wl.n_ch)[0].sum())
    sets = [(J2, par, inputs.enumerate_3n_channels(J2, par, 1, 3)) for J2 in range(1, 19, 2) for par in (+1, -1)]
    handles = [api.pm_lattice_attach(lat.h, ch, J2, par, 1, inputs.PM_FERMION_ISOSPIN) for J2, par, ch in sets]
    cap = hits * max(int(api.pm_lattice_coupling(h, len(ch))[0].sum()) for h, (_, _, ch) in zip(handles, sets))
    ci = torch.empty(cap, dtype=torch.int32, device="cuda")
    v = torch.empty(cap, dtype=torch.float64, device="cuda")
    rows, total_ms, total_nnz = [], 0.0, 0
    for h, (J2, par, ch) in zip(handles, sets):
        rpj = rp[: wl.n_cells * len(ch) + 1]
        api.pm_build_reuse(h, 0, wl.n_cells, rpj, ci, v)                 # untimed: run-time compilation of the set's kernel, if any
        flush.zero_()
        e0.record(st)
        n = api.pm_build_reuse(h, 0, wl.n_cells, rpj, ci, v)
        e1.record(st); torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        rows.append({"J2": J2, "parity": par, "channels": len(ch), "nnz": n, "ms": ms, "kernel": api.pm_lattice_fill_kernel(h)})
        total_ms += ms; total_nnz += n
        api.pm_lattice_destroy(h)
    del ci, v, rp
    torch.cuda.empty_cache()
    return {"what": f"all 18 J^pi <= 17/2, pair j <= 3, T = 1/2 on {wl.name}'s grid; pattern pass once + one pm_build_reuse per J^pi",
            "pattern_ms_once": pattern_ms, "fill_ms_total": total_ms, "total_ms": pattern_ms + total_ms, "total_nnz": total_nnz,
            "nnz_per_s": total_nnz / ((pattern_ms + total_ms) * 1e-3), "max_channels": max(r["channels"] for r in rows),
            "csr_bytes_largest": 12 * max(r["nnz"] for r in rows), "sets": rows}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="pm")
    ap.add_argument("--config", default="4", help="BASELINE.json configs index (default 4, the metric's workload)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-lattices", action="store_true", help="skip the five-lattice table")
    ap.add_argument("--sweep", action="store_true", help="also time the sweep over all J^pi <= 17/2 (62 channels) on the workload's grid")
    ap.add_argument("--e2e-steps", type=int, default=2)
    args = ap.parse_args()
    args.config = int(args.config)
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_1508_07441_b200 import api

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    # explicit build step (no-op when libpm.so is newer than its sources); local rank 0 builds, the others wait for it
    from paper_1508_07441_b200.csrc import build as lib_build
    if local == 0:
        lib_build.build()
    else:
        t_wait = time.time()
        while lib_build.stale() and time.time() - t_wait < 600:
            time.sleep(1.0)
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    api.lib()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    wl = inputs.config(args.config)
    lat = api.Lattice(wl)
    st = torch.cuda.current_stream()
    pk = _peaks()
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    # ---- the partition: one count pass over the lattice (every rank the same), contiguous cell ranges balanced by hits
    t0 = time.perf_counter()
    rp_all = torch.empty(wl.M + 1, dtype=torch.int64, device="cuda")
    nnz_total = api.pm_pattern(lat.h, 0, wl.n_cells, rp_all, None)
    hits = api.pm_pattern_cell_hits(lat.h, wl.n_cells)
    cuts, cell_cost = shard_cuts(api, hits, world)
    partition_ms = (time.perf_counter() - t0) * 1e3
    cb, ce = int(cuts[rank]), int(cuts[rank + 1])
    nnz_mine = int(hits[cb:ce].astype(np.int64).sum()) * int(nnz_total // max(1, int(hits.astype(np.int64).sum())))
    del rp_all
    # outputs allocated once (caller-owned buffers); every step rewrites them completely
    rowptr = torch.empty((ce - cb) * wl.n_ch + 1, dtype=torch.int64, device="cuda")
    colidx = torch.empty(max(nnz_mine, 1), dtype=torch.int32, device="cuda")
    vals = torch.empty(max(nnz_mine, 1), dtype=torch.float64, device="cuda")

    clocks = ClockSampler(local)
    step_ms, fill_ms, nnz_r, launches = timed_builds(api, torch, lat, wl, cb, ce, rowptr, colidx, vals, flush, args.steps, args.warmup,
                                                      world, barrier, st, clocks)
    assert nnz_r == nnz_mine, (nnz_r, nnz_mine)
    total_ms = max_over_ranks(sum(step_ms), world)
    value = job_throughput(nnz_total, args.steps, total_ms)
    nnz = nnz_total

    if world > 1:
        # sharded run: the headline line only (per-kernel analysis, e2e and the CPU baseline are 1-GPU measurements)
        fill_max = max_over_ranks(float(np.mean(fill_ms)), world)
        nnz_ranks = gather_counts(nnz_mine, world)
        if rank == 0:
            out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                   "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
                   "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                   "config": {"workload": wl.name, "M": wl.M, "n_channels": wl.n_ch, "cells": wl.n_cells,
                              "nodes_per_cell": wl.nodes_per_cell, "nnz": nnz_total, "csr_bytes": 12 * nnz_total,
                              "l2": "256 MiB buffer written between timed steps (L2 flush); outputs (12 B/nnz) exceed L2",
                              "sharding": "one lattice split over the ranks: contiguous source-cell ranges balanced by hit count "
                                          "(pm_partition_cells), each rank runs pm_build on its range, one all-gather of the per-rank nnz "
                                          "(8 B) per step turns block-local row pointers into global ones",
                              "cuts": [int(c) for c in cuts], "nnz_per_rank": nnz_ranks, "cell_cost": cell_cost,
                              "partition_ms_once": partition_ms},
                   "build_ms": {"best": float(np.min(step_ms)), "median": float(np.median(step_ms)), "fill_slowest_rank": fill_max},
                   "e2e": None, "cpu_baseline": None, "roofline": None, "gpu_launches": int(launches), "clocks": clocks.summary()}
            print(json.dumps(out))
        lat.close()
        dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the fill)
    dfma = api.pm_diag_dfma_tflops()
    roof = fill_roofline(api, lat, wl, nnz, fill_ms, pk, n_sm, dfma)

    # ---- the SpMV check (row a9): y = P0 x on the matrix just built; HBM bound, 12 B per nonzero
    xv = torch.rand(wl.M, dtype=torch.float64, device="cuda")
    yv = torch.empty(wl.M, dtype=torch.float64, device="cuda")

    def best_of(fn, n=6):
        ms = []
        for it in range(n):
            flush.zero_()
            s0, s1 = (torch.cuda.Event(enable_timing=True) for _ in range(2))
            s0.record(st)
            fn()
            s1.record(st)
            torch.cuda.synchronize()
            if it:
                ms.append(s0.elapsed_time(s1))
        return min(ms)

    spmv_ms = best_of(lambda: api.pm_spmv(lat.h, rowptr, colidx, vals, xv, yv))
    spmv_gbs = 12.0 * nnz / (spmv_ms * 1e-3) * 1e-9
    spmv = {"ms": spmv_ms, "bound": "hbm", "achieved": spmv_gbs, "peak": pk["hbm_gbs"], "unit": "GB/s",
            "frac": spmv_gbs / pk["hbm_gbs"]}
    # ---- the iteration step K u = O P0 V~1 G1 u (eq. 24) with seeded synthetic factors
    O_, V1_, g1_, u_ = inputs.iteration_factors(wl)
    Vt_ = np.stack([O_[a].T @ V1_[a] for a in range(wl.n_ch)])           # caller-side input preparation
    dO, dVt, dg, du = (torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (O_, Vt_, g1_, u_))
    work = torch.empty(2 * wl.M, dtype=torch.float64, device="cuda")
    it_ms = best_of(lambda: api.pm_kernel_apply(lat.h, rowptr, None, vals, dO, dVt, dg, du, yv, work))     # columns implied by the hit lists
    it_gbs = 8.0 * nnz / (it_ms * 1e-3) * 1e-9
    iteration = {"ms": it_ms, "bound": "hbm", "achieved": it_gbs, "peak": pk["hbm_gbs"], "unit": "GB/s",
                 "frac": it_gbs / pk["hbm_gbs"],
                 "what": "K u = O P0 V~1 G1 u, synthetic O, V1, G1 (seed 2025), SpMV without the column array; "
                         "bytes = 8 B per nonzero of P0 (with the column array: 12 B and the time of `spmv` + 0.15 ms)"}
    rot_ms = best_of(lambda: api.pm_rotate_apply(lat.h, rowptr, None, vals, dO, du, yv, work))
    rotation = {"ms": rot_ms, "bound": "hbm", "achieved": 8.0 * nnz / (rot_ms * 1e-3) * 1e-9, "peak": pk["hbm_gbs"], "unit": "GB/s",
                "frac": 8.0 * nnz / (rot_ms * 1e-3) * 1e-9 / pk["hbm_gbs"], "what": "P x = O P0 O^T x (eq. 20), same synthetic O"}
    # ---- the operator form of P0 (per-pair sums): build, apply, and the iteration step through it
    operator = None
    try:
        e0, e1 = (torch.cuda.Event(enable_timing=True) for _ in range(2))
        api.pm_operator_build(lat.h)                                     # untimed: run-time compilation of the sums kernel
        flush.zero_()
        e0.record(st)
        pairs, op_bytes = api.pm_operator_build(lat.h)
        e1.record(st); torch.cuda.synchronize()
        op_build_ms = e0.elapsed_time(e1)
        op_ms = best_of(lambda: api.pm_operator_apply(lat.h, xv, yv))
        ref = torch.empty_like(yv)
        api.pm_spmv(lat.h, rowptr, colidx, vals, xv, ref)
        api.pm_operator_apply(lat.h, xv, yv)
        op_err = float((yv - ref).abs().max() / ref.abs().max())
        w1, w2 = work[: wl.M], work[wl.M:]

        def op_iteration():                                             # K u = O (P0 (V~1 (G1 u))), P0 applied from the sums
            api.pm_block_apply(lat.h, dVt, dg, du, w1)
            api.pm_operator_apply(lat.h, w1, w2)
            api.pm_block_apply(lat.h, dO, None, w2, yv)
        op_it_ms = best_of(op_iteration)
        operator = {"pairs": pairs, "bytes": op_bytes, "csr_value_bytes": 8 * nnz, "build_ms": op_build_ms, "apply_ms": op_ms,
                    "apply_gbs": op_bytes / (op_ms * 1e-3) * 1e-9, "apply_frac_of_hbm": op_bytes / (op_ms * 1e-3) * 1e-9 / pk["hbm_gbs"],
                    "iteration_ms": op_it_ms, "max_rel_diff_vs_spmv": op_err,
                    "what": "per-pair sums of the orbital functions (pm_operator_build) and y = P0 x straight from them (pm_operator_apply)"}
    except Exception as ex:                                              # (needs NVRTC on the box)
        operator = {"error": repr(ex)}
    del xv, yv, work

    # ---- the five lattices (north_star): device-timed pm_build of each, same timing rules
    lattices = None
    if not args.no_lattices:
        lattices = []
        for k in range(5):
            if k == args.config:
                lattices.append({"config": k, "workload": wl.name, "M": wl.M, "nnz": nnz, "ms_per_build": float(np.median(step_ms)),
                                 "nnz_per_s": nnz / (float(np.median(step_ms)) * 1e-3), "fill_ms": float(np.median(fill_ms)),
                                 "hbm_frac": roof["hbm"]["frac"], "alu_frac": roof["alu"]["frac"], "bound": roof["bound"]})
                continue
            wk = inputs.config(k)
            lk = api.Lattice(wk)
            rpk = torch.empty(wk.M + 1, dtype=torch.int64, device="cuda")
            nk = api.pm_pattern(lk.h, 0, wk.n_cells, rpk, None)
            cik = torch.empty(nk, dtype=torch.int32, device="cuda"); vk = torch.empty(nk, dtype=torch.float64, device="cuda")
            sm, fm, _, _ = timed_builds(api, torch, lk, wk, 0, wk.n_cells, rpk, cik, vk, flush, 5, 3, 1, barrier, st)
            rk = fill_roofline(api, lk, wk, nk, fm, pk, n_sm, None)
            lattices.append({"config": k, "workload": wk.name, "M": wk.M, "nnz": nk, "ms_per_build": float(np.median(sm)),
                             "nnz_per_s": nk / (float(np.median(sm)) * 1e-3), "fill_ms": float(np.median(fm)),
                             "hbm_frac": rk["hbm"]["frac"], "alu_frac": rk["alu"]["frac"], "bound": rk["bound"]})
            lk.close()
            del rpk, cik, vk

    # ---- every J^pi <= 17/2 on this grid (on request: ~70 GB of device buffers, ~25 s)
    sweep = None
    if args.sweep:
        colidx = vals = None                                     # (the sweep needs ~70 GB of its own)
        torch.cuda.empty_cache()
        try:
            sweep = jpi_sweep(api, torch, lat, wl, flush, st)
        except Exception as ex:                                  # the headline line must not depend on it
            sweep = {"error": repr(ex)}
            print("sweep failed:", repr(ex), file=sys.stderr)
        torch.cuda.empty_cache()

    # ---- end to end through the C ABI with HOST buffers (D2H copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        h_rp = torch.empty(wl.M + 1, dtype=torch.int64, pin_memory=True)
        h_ci = torch.empty(nnz, dtype=torch.int32, pin_memory=True)
        h_v = torch.empty(nnz, dtype=torch.float64, pin_memory=True)
        colidx = vals = None
        torch.cuda.empty_cache()

        def e2e_step():
            # the call a user makes: create the lattice from host arrays (host precompute + table upload),
            # build with host outputs (pattern, fill and device->host copies), destroy
            l2 = api.Lattice(wl)
            r = api.pm_build_host(l2.h, 0, h_rp, h_ci, h_v)
            l2.close()
            return r

        e2e_step()
        barrier()
        t0 = time.perf_counter()
        nb = 1
        for _ in range(args.e2e_steps):
            _, nb = e2e_step()
        barrier()
        dt_s = time.perf_counter() - t0
        h2d = wl.p_edges.nbytes + wl.q_edges.nbytes + wl.channels.nbytes + sum(a.nbytes + b.nbytes for a, b in wl.rules.values())
        e2e = {"value": job_throughput(nnz, args.e2e_steps, dt_s * 1e3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(12 * nnz + 8 * (wl.M + 1)), "blocks": nb, "steps": args.e2e_steps,
               "api": "pm_lattice_create + pm_lattice_set_rule + pm_build_host (pinned host buffers) + pm_lattice_destroy"}

    cpu = None
    if not args.no_cpu:
        cpu = cpu_baseline(wl)
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
           "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": wl.name, "M": wl.M, "n_channels": wl.n_ch, "cells": wl.n_cells,
                      "nodes_per_cell": wl.nodes_per_cell, "nnz": nnz, "csr_bytes": 12 * nnz, "blocks": 1,
                      "l2": "256 MiB buffer written between timed steps (L2 flush); outputs (12 B/nnz) exceed L2",
                      "sharding": "N > 1: one lattice split over the ranks by source-cell ranges (strong scaling); N = 1: the whole lattice"},
           "build_ms": {"best": float(np.min(step_ms)), "median": float(np.median(step_ms)),
                        "pattern_median": float(np.median(np.array(step_ms) - np.array(fill_ms))),
                        "fill_median": float(np.median(fill_ms)), "fill_best": float(np.min(fill_ms)),
                        "fill_all": [round(float(x), 3) for x in fill_ms]},
           "roofline": roof, "spmv": spmv, "iteration": iteration, "rotation": rotation, "operator": operator, "lattices": lattices, "sweep": sweep,
           "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks.summary()}
    print(json.dumps(out))
    lat.close()


if __name__ == "__main__":
    main()
