"""One-off checks at sizes and densities the pytest suite does not reach (run by hand on a B200; not collected by pytest):

    python tests/large_inputs_check.py --n 16777216            # uniform LJ-like fluid, r = 1.5, capacity 32
    python tests/large_inputs_check.py --n 1048576 --droplet 64   # all particles in 1/64 of the box volume

Builds and traverses through the C-ABI binding, times both with CUDA events (best of `--reps`), and compares the
per-particle neighbor counts with the CPU oracle's cell list (exact; rows beyond the capacity are compared by count
only).  Prints one JSON line.  PAPER.md:212-214 (strongly inhomogeneous systems), PAPER.md:186 (large N)."""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def make(N, droplet, rho, seed):
    """Ideal-gas positions at density rho, in the whole box (droplet = 1) or in a cube of 1/droplet of its volume."""
    from paper_1901_08088_b200 import workloads as W
    rng = np.random.default_rng([4242, seed])
    side = (N / rho) ** (1.0 / 3.0)                  # edge of the region that holds the particles
    L = side * droplet ** (1.0 / 3.0)                # edge of the box
    p = rng.random((N, 3)) * side + 0.5 * (L - side)
    return W._finish(p, L)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=1 << 24)
    ap.add_argument("--droplet", type=int, default=1)
    ap.add_argument("--rho", type=float, default=0.85)
    ap.add_argument("--r", type=float, default=1.5)
    ap.add_argument("--cap", type=int, default=32)
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--cell-level", type=int, default=0, help="QBVH_OPT_CELL_LEVEL (0: chosen from N)")
    ap.add_argument("--group-max", type=int, default=32, help="QBVH_OPT_GROUP_MAX")
    ap.add_argument("--stats", action="store_true", help="one more, instrumented traversal: counters of the production kernel")
    ap.add_argument("--config", type=int, default=0, help="a BASELINE.json config (full size) instead of the ideal gas")
    ap.add_argument("--no-oracle", action="store_true")
    a = ap.parse_args()
    import torch
    from paper_1901_08088_b200 import qbvh
    dev = torch.device("cuda:0")
    if a.config:
        from paper_1901_08088_b200 import workloads as W
        w = W.make_config(a.config)
        assert w.T == 1, "single-type configs only"
        pos, box, r_list = w.pos, w.box, w.r_list
        a.n, a.cap, a.r = w.N, w.max_neigh, float(w.r_list[0, 0])
    else:
        pos, box = make(a.n, a.droplet, a.rho, 0)
        r_list = np.array([[a.r]], np.float32)
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, 32)
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
    qbvh.qbvh_set_option(qbvh.OPT_CELL_LEVEL, a.cell_level)
    qbvh.qbvh_set_option(qbvh.OPT_GROUP_MAX, a.group_max)
    nl = qbvh.NeighborList(a.n, T=1, max_neigh=a.cap, device=dev)
    dpos = torch.from_numpy(pos).to(dev)
    tb, tt, M = [], [], 0
    for _ in range(a.reps + 1):
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        e[0].record()
        nl.build(dpos, None, box)
        e[1].record()
        nl.neighbors_enqueue(r_list)
        e[2].record()
        M = nl.neighbors_result()
        torch.cuda.synchronize()
        tb.append(e[0].elapsed_time(e[1]))
        tt.append(e[1].elapsed_time(e[2]))
    counts = qbvh.qbvh_debug_export(qbvh.EXPORT_COUNTS, a.n)
    n_gpu = nl.n_neigh[: a.n].cpu().numpy()
    out = {"N": a.n, "droplet": a.droplet, "rho": a.rho, "r": a.r, "cap": a.cap, "box_L": float(box[3]),
           "build_ms": min(tb[1:]), "traverse_ms": min(tt[1:]), "M": int(M), "nn": float(n_gpu.mean()),
           "cell_level": int(counts[3]), "cells": int(counts[2]), "groups": int(counts[1]),
           "workspace_GB": qbvh.qbvh_workspace_bytes(a.n, 1) / 1e9, "group_max": a.group_max}
    if a.stats:
        qbvh.qbvh_set_option(qbvh.OPT_STATS, 1)
        nl.neighbors(r_list, retry=False)
        st = qbvh.qbvh_get_stats()
        qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
        out.update(lanes_per_group=a.n / max(st["groups"], 1), candidates_per_group=st["group_candidates"] / max(st["groups"], 1),
                   dist_checks_per_particle=st["group_dist_checks"] / a.n, node_tests_per_group=st["group_node_tests"] / max(st["groups"], 1),
                   walk_steps_per_group=st["group_walk_steps"] / max(st["groups"], 1),
                   check_lane_slots_per_particle=32.0 * st["group_candidates"] / a.n)
    if not a.no_oracle:
        from oracle import neighbors as ON
        t0 = time.perf_counter()
        rp, nb, _ = ON.neighbor_list(pos, None, box, r_list, method="cell", with_band=False)
        out["oracle_s"] = time.perf_counter() - t0
        n_or = np.diff(rp)
        out["counts_equal"] = bool(np.array_equal(n_gpu, n_or))
        out["M_equal"] = bool(M == int(n_or.max()))
        # rows that fit: the sets themselves, on a sample of 200,000 rows
        rows = np.random.default_rng(1).choice(a.n, size=min(a.n, 200_000), replace=False)
        lst = nl.nlist[torch.from_numpy(rows).to(dev)].cpu().numpy()
        bad = 0
        for k, i in enumerate(rows):
            if n_or[i] <= a.cap:
                bad += not np.array_equal(np.sort(lst[k, : n_or[i]]), nb[rp[i]:rp[i + 1]])
        out["sampled_rows"] = int(len(rows))
        out["sampled_rows_mismatched"] = int(bad)
    print(json.dumps(out))


if __name__ == "__main__":
    main()
