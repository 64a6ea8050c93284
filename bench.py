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
KERNELS_PER_STEP = 7    # morton_hist (+finalize in its last block), 4 x onesweep, tree (hierarchy+fit+quantize), traverse_group


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
    if cid == 2:
        return W.lj_lattice(N=131072, n_lat=51), "config-2 recipe at N=131,072 (n_lat=51), same density/jitter/cutoff"
    w = W.make_config(cid, small=True)
    return w, f"config-{cid} recipe at reduced size N={w.N}"


def time_oracle(w, repeats: int = 1):
    from oracle import neighbors as ON
    best = None
    for _ in range(repeats):
        t = {}
        ON.neighbor_list(w.pos, w.type, w.box, w.r_list, method="cell", with_band=False, timing=t)
        best = t if best is None or t["seconds"] < best["seconds"] else best
    return best


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
            "config": {"workload": f"BASELINE.json configs[{args.config - 1}] (bounded sample: {what})",
                       "N_sample": w.N},
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
    nl = qbvh.NeighborList(N, T=T, max_neigh=cap, device=dev)
    pos = torch.from_numpy(w.pos).to(dev)
    typ = None if w.type is None else torch.from_numpy(w.type).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def step():
        nl.build(pos, typ, w.box)
        return nl.neighbors(w.r_list, retry=False)

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
        nl.build(pos, typ, w.box)
        ev[s][1].record()
        nl.neighbors(w.r_list, retry=False)
        ev[s][2].record()
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
    nl.neighbors(w.r_list, retry=False)
    stats = qbvh.qbvh_get_stats()
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
    nn = stats["neighbors"] / N

    # ---- end to end through the HOST-buffer C-ABI calls ----
    e2e_ms = None
    if not args.no_e2e:
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
        qbvh.qbvh_set_staging(None)
    clocks = sampler.stop()
    h2d = 12 * N + (4 * N if w.type is not None else 0)
    d2h = 4 * N * cap + 4 * N + 8

    # ---- roofline of the dominant kernel (traverse_kernel), algorithmic bytes per SURVEY.md §8(d) ----
    peak, peak_src = measured_peaks()
    trav_bytes = N * (52.0 + 4.0 * nn)
    build_bytes = N * (188.0 + (4.0 if w.type is not None else 0.0))
    trav_ms, build_ms = float(np.mean(t_trav)), float(np.mean(t_build))
    ach = trav_bytes / (trav_ms * 1e-3) / 1e9
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traverse_traffic_bytes.txt")
    if os.path.exists(tp):
        try:
            traffic = float(open(tp).read().split()[0])
        except Exception:
            traffic = None
    roofline = {"bound": "hbm", "kernel": "traverse_group_kernel", "achieved": ach, "peak": peak, "unit": "GB/s",
                "frac": ach / peak, "traffic": traffic, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": trav_bytes}
    # plain-ALU view of the same kernel: thread-instructions issued / (148 SM x 128 lanes x f)
    whole = (trav_bytes + build_bytes) / (ms_per_step * 1e-3) / 1e9

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config - 1}]: {w.name}", "N": N, "types": T,
                       "r_list": [float(x) for x in np.asarray(w.r_list).reshape(-1)], "max_neigh": cap,
                       "leaf_collapse": args.leaf_collapse, "l2": "flushed between timed iterations (256 MiB memset)",
                       "parallelism": "replicas" if world > 1 else "single GPU"},
            "build_ms": build_ms, "traverse_ms": trav_ms,
            "build_ns_per_particle": 1e6 * build_ms / N, "traverse_ns_per_particle": 1e6 * trav_ms / N,
            "neighbors_per_particle": nn, "max_neighbors": int(M),
            "dist_checks_per_s": stats["dist_checks"] / (trav_ms * 1e-3),
            "node_tests_per_particle": stats["node_tests"] / N, "dist_checks_per_particle": stats["dist_checks"] / N,
            "roofline": roofline,
            "roofline_whole_path": {"bound": "hbm", "achieved": whole, "peak": peak, "unit": "GB/s", "frac": whole / peak,
                                    "algorithmic_bytes_per_step": trav_bytes + build_bytes},
            "e2e": (None if e2e_ms is None else
                    {"value": 1e6 * e2e_ms / (N * world), "unit": UNIT, "ms_per_step": e2e_ms,
                     "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": Ke}),
            "gpu_launches": KERNELS_PER_STEP * K, "clocks": clocks, "wall_s_timed_loop": wall}

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        ws, what = (w, "the full workload, one pass (best of 2)") if N <= (1 << 21) else reference_sample(args.config)
        t = time_oracle(ws, repeats=2)
        line["cpu_baseline"] = {"value": 1e9 * t["seconds"] / ws.N, "unit": UNIT, "cores": t["threads"],
                                "kind": "oracle", "sample": what, "seconds": t["seconds"]}
    if rank == 0:
        print(json.dumps(line))
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
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg (profiling runs)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
