#!/usr/bin/env python
"""bench.py — headline benchmark: quantized-BVH neighbor list, build + traverse, ns/particle at 1M LJ (config 2).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl reference]

One "step" = one pass of the whole hot path (qbvh_build + qbvh_neighbors) over the
seeded synthetic config-2 workload (BASELINE.json configs[1]).  Prints ONE JSON line.  Multi-GPU = independent
replicas (the path runs on one GPU; no data-path collective), weak scaling.
`--impl reference` times the CPU oracle (the only other place that may execute oracle/).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "neighbor-list build+traverse ns/particle at 1M LJ"
UNIT = "ns/particle"
KERNELS_PER_STEP = 6    # morton_cell, cell_scan, cell_scatter, cell_tree, top_tree, traverse_group


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.005):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.sm_max = [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
                 "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=1.0)
        med = int(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def max_over_ranks(value: float, world: int, device=None) -> float:
    """Timing of a multi-rank run = the slowest rank (replicas: no other exchange on the path)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    tt = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def whole_job_value(ms_per_step: float, n_per_rank: int, world: int) -> float:
    """ns per particle of the whole job: all ranks' particles over the slowest rank's time."""
    return 1e6 * ms_per_step / (n_per_rank * world)


def reference_sample(cid: int):
    """Bounded sample of the workload for the oracle arm: same recipe, density, cutoff; fewer particles."""
    from paper_1901_08088_b200 import workloads as W
    if cid in (1, 2):
        w = W.make_config(cid)
        return w, f"the full workload (N={w.N}), one pass of the cell-list oracle per step"
    w = W.make_config(cid, small=True)
    return w, f"config-{cid} recipe at reduced size N={w.N}"


def omp_threads(n: int | None = None) -> int:
    """Thread count of the OpenMP runtime the oracle runs on (libgomp, shared with liboracle.so); sets it when n is given."""
    import ctypes
    gomp = ctypes.CDLL("libgomp.so.1")
    prev = int(gomp.omp_get_max_threads())
    if n is not None:
        gomp.omp_set_num_threads(int(n))
    return prev


def time_oracle(w, repeats: int = 1, threads: int | None = None):
    """The oracle as it stands, timed on the host cores (all of them, or `threads`)."""
    from oracle import neighbors as ON
    best = None
    prev = omp_threads(threads) if threads is not None else None
    try:
        for _ in range(repeats):
            t = {}
            ON.neighbor_list(w.pos, w.type, w.box, w.r_list, method="cell", with_band=False, timing=t)
            best = t if best is None or t["seconds"] < best["seconds"] else best
    finally:
        if prev is not None:
            omp_threads(prev)
    return best


def config_keys(cid: int, w) -> dict:
    """The workload description both arms print (identical keys and values for the same --config)."""
    return {"workload": f"BASELINE.json configs[{cid - 1}]: {w.name}", "N": w.N, "types": w.T,
            "r_list": [float(x) for x in np.asarray(w.r_list).reshape(-1)], "max_neigh": w.max_neigh}


def aabb_census(w, nl, qbvh, torch, dev):
    """'Extra false-positive AABB tests' of the quantized tree (north_star): Algorithm 1's
    node tests and leaf overlaps per particle on the quantized one-particle-per-leaf tree — counted by the GPU census
    (QBVH_OPT_STATS, K = 1) — against the same walk on the tree's unquantized fp32 boxes, counted by the oracle replay
    (the library keeps no fp32 boxes).  Outside every timed region."""
    from oracle import tree as OT
    K0 = qbvh.qbvh_get_option(qbvh.OPT_LEAF_COLLAPSE)
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, 1)
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 1)
    try:
        nl.build(torch.from_numpy(w.pos).to(dev), None if w.type is None else torch.from_numpy(w.type).to(dev), w.box)
        nl.neighbors(w.r_list, retry=False)
        s = qbvh.qbvh_get_stats()
    finally:
        qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
        qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, K0)
    t = OT.build(w.pos, w.type, w.box, T=w.T)
    f = OT.traverse_fp32_boxes(t, w.box, w.r_list)
    N = w.N
    tq, tf = s["node_tests"] / N, float(f["n_tests"].sum()) / N
    lq, lf = s["leaf_overlaps"] / N, float(f["n_overlap"].sum()) / N
    return {"node_tests_per_particle_quantized": tq, "node_tests_per_particle_fp32_boxes": tf,
            "extra_node_tests_per_particle": tq - tf, "extra_node_tests_frac": (tq - tf) / tf if tf else None,
            "leaf_overlaps_per_particle_quantized": lq, "leaf_overlaps_per_particle_fp32_boxes": lf,
            "extra_leaf_overlaps_per_particle": lq - lf,
            "source": "quantized: GPU census (QBVH_OPT_STATS, leaf collapse 1); fp32 boxes: oracle replay on the same tree"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w, what = reference_sample(args.config)
    for _ in range(args.warmup):
        time_oracle(w)
    t0 = time.perf_counter()
    threads = 1
    for _ in range(args.steps):
        threads = time_oracle(w)["threads"]
    dt = time.perf_counter() - t0
    ms = 1e3 * dt / max(args.steps, 1)
    val = 1e6 * ms / w.N
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": config_keys(args.config, w), "notes": {"sample": what},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": what},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_1901_08088_b200 import qbvh
    from paper_1901_08088_b200 import workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    w = W.make_config(args.config, seed=rank)          # replicas: each rank its own seeded configuration
    N, T, cap = w.N, w.T, w.max_neigh
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, args.leaf_collapse)
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
    if args.variant is not None:
        qbvh.qbvh_set_option(qbvh.OPT_VARIANT, args.variant)
    nl = qbvh.NeighborList(N, T=T, max_neigh=cap, device=dev)
    f64 = args.dtype == "f64"
    if f64:                                            # fp64 particles, fp32 tree (an extra, not the headline)
        pos64, box, r_list = W.as_f64(w, seed=rank)
        pos = torch.from_numpy(pos64).to(dev)
    else:
        pos, box, r_list = torch.from_numpy(w.pos).to(dev), w.box, w.r_list
    typ = None if w.type is None else torch.from_numpy(w.type).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def step():
        nl.build(pos, typ, box)
        return nl.neighbors(r_list, retry=False)

    M = 0
    for _ in range(max(args.warmup, 3)):
        M = step()
    if M > cap:
        raise SystemExit(f"max_neigh={cap} overflows (M={M}); no retry inside the timed loop")
    torch.cuda.synchronize()

    K = args.steps
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]
    sampler = ClockSampler(local)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.start()
    wall0 = time.perf_counter()
    for s in range(K):
        flush.zero_()                                  # L2 flush between timed iterations (outside the events)
        ev[s][0].record()
        nl.build(pos, typ, box)
        ev[s][1].record()
        # the traversal is enqueued (fp32 or fp64 form), the closing event recorded behind it on the stream, and only then
        # does the host wait for M: the events bracket the device work, not the host's wake-up after the synchronise
        nl.neighbors_enqueue(r_list)
        ev[s][2].record()
        if nl.neighbors_result() > cap:
            raise SystemExit("overflow inside the timed loop")
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    if world > 1:
        dist.barrier()
    t_build = np.array([e[0].elapsed_time(e[1]) for e in ev])
    t_trav = np.array([e[1].elapsed_time(e[2]) for e in ev])
    total_ms = max_over_ranks(float((t_build + t_trav).sum()), world, dev)
    ms_per_step = total_ms / K
    value = whole_job_value(ms_per_step, N, world)     # ns per particle, whole job

    # ---- statistics of the run (one instrumented pass, outside the timed region) ----
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 1)
    nl.neighbors(r_list, retry=False)
    stats = qbvh.qbvh_get_stats()
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
    nn = float(nl.n_neigh[:N].sum().item()) / N
    counts = qbvh.qbvh_debug_export(qbvh.EXPORT_COUNTS, N)      # nodes written, query groups, cells, cell level

    # ---- end to end through the HOST-buffer C-ABI calls ----
    e2e_ms = None
    d2h = 0
    if not args.no_e2e and not f64:
        stg = torch.empty(qbvh.qbvh_staging_bytes(N, cap), dtype=torch.uint8, device=dev)
        qbvh.qbvh_set_staging(stg)
        hpos = torch.from_numpy(w.pos).pin_memory()
        htyp = None if w.type is None else torch.from_numpy(w.type).pin_memory()
        hlist = torch.empty((N, cap), dtype=torch.int32).pin_memory()
        hcnt = torch.empty(N, dtype=torch.int32).pin_memory()
        Ke = max(3, min(K, 10))
        for _ in range(2):
            qbvh.qbvh_build_host(hpos, htyp, N, w.box)
            qbvh.qbvh_neighbors_host(w.r_list, hlist, hcnt, cap)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(Ke):
            qbvh.qbvh_build_host(hpos, htyp, N, w.box)
            qbvh.qbvh_neighbors_host(w.r_list, hlist, hcnt, cap)
        e1.record()
        torch.cuda.synchronize()
        e2e_ms = e0.elapsed_time(e1) / Ke
        e2e_ms = max_over_ranks(e2e_ms, world, dev)
        d2h = qbvh.qbvh_last_d2h_bytes()               # n_neigh + the min(M, max_neigh) columns actually copied + 8
        qbvh.qbvh_set_staging(None)
    clocks = sampler.stop()
    h2d = 12 * N + (4 * N if w.type is not None else 0)

    # ---- roofline of the dominant kernel (traverse_kernel), algorithmic bytes per SURVEY.md §8(d) ----
    peak, peak_src = measured_peaks()
    trav_bytes = N * (52.0 + 4.0 * nn)
    build_bytes = N * (188.0 + (4.0 if w.type is not None else 0.0))
    trav_ms, build_ms = float(np.mean(t_trav)), float(np.mean(t_build))
    ach = trav_bytes / (trav_ms * 1e-3) / 1e9
    # Counters of one traversal launch that only a profiler sees: STORED ncu measurements (profiles/), valid for
    # config 2 / fp32 at the commit named beside them; null for anything else.
    traffic = traffic_commit = None
    counters = {}
    tp = os.path.join(ROOT, "profiles", "traverse_ncu_counters.txt")
    if os.path.exists(tp) and args.config == 2 and not f64:
        try:
            counters = dict(tok.split("=", 1) for tok in open(tp).read().split() if "=" in tok)
            traffic, traffic_commit = float(counters["dram_bytes"]), counters.get("commit")
        except Exception:
            traffic = traffic_commit = None
            counters = {}
    roofline = {"bound": "hbm", "kernel": "traverse_group_kernel", "achieved": ach, "peak": peak, "unit": "GB/s",
                "frac": ach / peak, "traffic": traffic, "traffic_source": "stored ncu capture", "traffic_commit": traffic_commit,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": trav_bytes}
    # What actually bounds the kernel is on-chip throughput, not bytes.  The profiler's own utilisation
    # figures of the stored capture (same commit stamp), quoted as they are — no derived "issue slot" arithmetic.
    roofline_issue = None
    if "inst_executed" in counters:
        def num(k):
            return float(counters[k]) if k in counters else None
        roofline_issue = {"kernel": "traverse_group_kernel", "source": "stored ncu capture (profiles/traverse_ncu_counters.txt)",
                          "commit": traffic_commit, "warp_instructions_per_launch": num("inst_executed"),
                          "warp_instructions_per_particle": num("inst_executed") / N,
                          "sm_issue_active_pct": num("issue_active_pct"),
                          "l1tex_lsu_data_pipe_wavefronts_pct": num("lsu_data_pipe_pct"),
                          "shared_wavefronts": num("shared_wavefronts"),
                          "shared_bank_conflict_wavefronts": num("shared_bank_conflicts")}
    roofline_build = {"bound": "hbm", "kernel": "build (morton_cell + cell_scan + cell_scatter + cell_tree + top_tree)",
                      "achieved": build_bytes / (build_ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                      "frac": build_bytes / (build_ms * 1e-3) / 1e9 / peak, "algorithmic_bytes_per_step": build_bytes}
    whole = (trav_bytes + build_bytes) / (ms_per_step * 1e-3) / 1e9

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64 particles / f32 tree" if f64 else "f32", "data": "synthetic",
            "config": config_keys(args.config, w),
            "notes": {"leaf_collapse": args.leaf_collapse, "l2": "flushed between timed iterations (256 MiB memset)",
                      "parallelism": "replicas" if world > 1 else "single GPU"},
            "build_ms": build_ms, "traverse_ms": trav_ms,
            "build_ns_per_particle": 1e6 * build_ms / N, "traverse_ns_per_particle": 1e6 * trav_ms / N,
            "neighbors_per_particle": nn, "max_neighbors": int(M),
            # the timed (production) kernel: pair-predicate evaluations and node tests of the group walk
            "dist_checks_per_s": stats["group_dist_checks"] / (trav_ms * 1e-3),
            "dist_checks_per_particle": stats["group_dist_checks"] / N,
            "node_tests_per_particle": stats["group_node_tests"] / N,
            # census of Algorithm 1 walked once per particle on the same tree (the paper's kernel; not the timed one)
            "census_node_tests_per_particle": stats["node_tests"] / N,
            "census_dist_checks_per_particle": stats["dist_checks"] / N,
            "nodes_written": int(counts[0]), "node_bytes": 16 * int(counts[0]), "node_bytes_uncollapsed": 16 * (2 * N - 1),
            "query_groups": int(counts[1]), "morton_cells": int(counts[2]), "cell_level": int(counts[3]),
            # how full the query groups are and how many pair checks a found neighbor costs (the decomposition's own overhead)
            "lanes_per_group": N / max(stats["groups"], 1),
            "candidates_per_neighbor": stats["group_dist_checks"] / max(nn * N, 1.0),
            "roofline": roofline, "roofline_issue": roofline_issue, "roofline_build": roofline_build,
            "roofline_whole_path": {"bound": "hbm", "achieved": whole, "peak": peak, "unit": "GB/s", "frac": whole / peak,
                                    "algorithmic_bytes_per_step": trav_bytes + build_bytes},
            "e2e": (None if e2e_ms is None else
                    {"value": 1e6 * e2e_ms / (N * world), "unit": UNIT, "ms_per_step": e2e_ms,
                     "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": Ke}),
            "gpu_launches": KERNELS_PER_STEP * K, "clocks": clocks, "wall_s_timed_loop": wall}

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        ws, what = (w, "the full workload, one pass (best of 2)") if N <= (1 << 21) else reference_sample(args.config)
        if f64:
            from oracle import neighbors as ON
            t = {}
            ON.neighbor_list_f64(pos64, w.type, box, r_list, method="cell", timing=t)
            what = "the full fp64 workload, one pass of the fp64 cell-list oracle"
        else:
            t = time_oracle(ws, repeats=2)
        line["cpu_baseline"] = {"value": 1e9 * t["seconds"] / ws.N, "unit": UNIT, "cores": t["threads"],
                                "kind": "oracle", "sample": what, "seconds": t["seconds"]}
        if not f64 and t["seconds"] * t["threads"] <= 25.0:          # bounded: about 10-30 s of CPU work at most
            t1 = time_oracle(ws, repeats=1, threads=1)       # "plus the 1-thread time"
            line["cpu_baseline"].update(value_1thread=1e9 * t1["seconds"] / ws.N, seconds_1thread=t1["seconds"])
        if not f64 and not args.no_census and N <= (1 << 21):
            line["aabb_tests"] = aabb_census(w, nl, qbvh, torch, dev)
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_sharded(args):
    """Strong-scaling extra (not the headline): the config's particles split over the ranks, one
    all-gather of positions per step (NCCL), the full build on every rank, the traversal of the rank's Z-order slice."""
    import torch
    import torch.distributed as dist
    from paper_1901_08088_b200 import qbvh, sharded
    from paper_1901_08088_b200 import workloads as W
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    w = W.make_config(args.config, seed=0)              # ONE system, the same on every rank
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, args.leaf_collapse)
    snl = sharded.ShardedNeighborList(w.N, T=w.T, max_neigh=w.max_neigh, device=dev)
    lo, cnt = snl.own_first, snl.own_count
    pos = torch.from_numpy(w.pos[lo:lo + cnt]).to(dev)
    typ = None if w.type is None else torch.from_numpy(w.type[lo:lo + cnt]).to(dev)
    nlist = torch.empty((max(snl.count, 1), w.max_neigh), dtype=torch.int32, device=dev)
    n_neigh = torch.zeros(max(snl.count, 1), dtype=torch.int32, device=dev)

    def step():
        snl.build(pos, typ, w.box)
        qbvh.qbvh_neighbors_range_enqueue(w.r_list, nlist, n_neigh, w.max_neigh, snl.first, snl.count)

    for _ in range(max(args.warmup, 3)):
        step()
        qbvh.qbvh_neighbors_result()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()                                        # behind the last traversal on the stream, before the host waits for it
    if qbvh.qbvh_neighbors_result() > w.max_neigh:
        raise SystemExit("overflow inside the timed loop")
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = max_over_ranks(e0.elapsed_time(e1) / args.steps, world, dev)
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": 1e6 * ms / w.N, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": False, "scaling": "strong",
                          "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                          "config": {"workload": f"BASELINE.json configs[{args.config - 1}]: {w.name}", "N": w.N,
                                     "parallelism": f"query sharding over {world} rank(s): all-gather of positions, full build per rank, Z-order slice per rank",
                                     "l2": "not flushed (back-to-back steps)"},
                          "gpu_launches": KERNELS_PER_STEP * args.steps}))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_slab(args):
    """Strong-scaling extra (SURVEY 8e bullet 2 / 8f NEXT-4 second half): slab decomposition with halos.  One system; rank g
    owns slab g along the longest axis; per step one neighbor exchange of the halo particles (NCCL P2P), the build over
    own + ghosts, the traversal, rows of the own particles mapped to global ids.  Nothing is redundant across ranks."""
    import torch
    import torch.distributed as dist
    from paper_1901_08088_b200 import qbvh, sharded
    from paper_1901_08088_b200 import workloads as W
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    w = W.make_config(args.config, seed=0)              # ONE system, the same on every rank
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, args.leaf_collapse)
    snl = sharded.SlabNeighborList(w.box, w.r_list, T=w.T, max_neigh=w.max_neigh, device=dev)
    mine = np.nonzero(sharded.slab_index(w.pos, w.box, world, snl.axis) == rank)[0]
    pos = torch.from_numpy(w.pos[mine]).to(dev)
    typ = None if w.type is None else torch.from_numpy(w.type[mine]).to(dev)
    gid = torch.from_numpy(mine.astype(np.int64)).to(dev)

    def step():
        snl.build(pos, typ, gid, w.N)
        return snl.neighbors()

    for _ in range(max(args.warmup, 3)):
        step()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = max_over_ranks(e0.elapsed_time(e1) / args.steps, world, dev)
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": 1e6 * ms / w.N, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": False, "scaling": "strong",
                          "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config_keys(args.config, w),
                          "notes": {"parallelism": f"slab decomposition over {world} rank(s) along axis {snl.axis}: halo exchange (P2P), build and traversal of own + ghost particles",
                                    "halo_width": snl.h, "own": int(len(mine)), "ghosts": snl.n_ghost, "halo_bytes_sent_per_step": snl.halo_bytes,
                                    "l2": "not flushed (back-to-back steps)", "includes": "host-side halo selection and the id mapping of the rows"},
                          "gpu_launches": KERNELS_PER_STEP * args.steps}))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number 1..5 (default 2: 1M LJ)")
    ap.add_argument("--impl", default="qbvh", choices=["qbvh", "reference"])
    ap.add_argument("--leaf-collapse", type=int, default=32)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-census", action="store_true", help="skip the quantized-vs-fp32 AABB test census (oracle replay on the host)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg (profiling runs)")
    ap.add_argument("--variant", type=int, default=None, help="traversal kernel (QBVH_OPT_VARIANT); default: the library's")
    ap.add_argument("--sharded", action="store_true", help="extra: query sharding over the ranks (strong scaling) instead of replicas")
    ap.add_argument("--slab", action="store_true", help="extra: slab decomposition with halos over the ranks (strong scaling)")
    ap.add_argument("--dtype", default="f32", choices=["f32", "f64"], help="f64: double-precision particles on the fp32 tree (an extra line)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.sharded:
        return run_sharded(args)
    if args.slab:
        return run_slab(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
