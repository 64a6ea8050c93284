"""ORACLE — TEST INFRASTRUCTURE ONLY.  `python -m oracle.census_report [--full]`

Prints the table of BASELINE.md §1a "extra false-positive AABB tests caused by quantization" (north_star; PAPER.md:85,
89, 196-198): Algorithm 1 replayed per particle on the one-particle-per-leaf tree, once on the quantized
16-byte nodes (oracle_traverse) and once on the same tree's unquantized fp32 boxes (oracle_traverse_fp32_boxes).
Calls only oracle/ and the seeded input generators.
"""
from __future__ import annotations

import sys

import numpy as np

from oracle import neighbors as ON
from oracle import tree as OT
from paper_1901_08088_b200 import workloads as W


def census(w):
    t = OT.build(w.pos, w.type, w.box, T=w.T)
    q = OT.traverse(t, w.box, w.r_list)
    f = OT.traverse_fp32_boxes(t, w.box, w.r_list)
    rp, _, _ = ON.neighbor_list(w.pos, w.type, w.box, w.r_list, with_band=False)
    N = w.N
    self_hits = sum(int(n) for a, n in enumerate(np.diff(t.seg)) if w.r_list[a, a] > 0)   # a particle's own leaf, once
    return {"N": N, "tq": q["n_tests"].sum() / N, "tf": f["n_tests"].sum() / N, "lq": q["n_overlap"].sum() / N,
            "lf": f["n_overlap"].sum() / N, "true": (rp[-1] + self_hits) / N}


def main(full: bool):
    rows = [(f"config {c} (reduced size)", W.make_config(c, small=True)) for c in (1, 2, 3, 4, 5)]
    rows += [("LJ shape N=128,000 rho=0.2 r_c=3.0 (PAPER.md:198)", W.lj_uniform(N=128_000, rho=0.2, r_list=3.0, config_id=100, max_neigh=160)),
             ("LJ shape N=128,000 rho=0.8 r_c=3.0 (PAPER.md:198)", W.lj_uniform(N=128_000, rho=0.8, r_list=3.0, config_id=100, max_neigh=160))]
    if full:
        rows += [("config 2, N=1,048,576", W.make_config(2))]
    print("| workload | N | node tests / particle: fp32 boxes | quantized | extra (%) | accepted leaves / particle: true neighbors + self (within r_list) | fp32 boxes (within r_pad) | quantized | extra from quantization |")
    print("|---|---|---|---|---|---|---|---|---|")
    for name, w in rows:
        c = census(w)
        print(f"| {name} | {c['N']} | {c['tf']:.2f} | {c['tq']:.2f} | {c['tq'] - c['tf']:.2f} ({100 * (c['tq'] - c['tf']) / c['tf']:.2f} %) | "
              f"{c['true']:.2f} | {c['lf']:.2f} | {c['lq']:.2f} | {c['lq'] - c['lf']:.2f} |")


if __name__ == "__main__":
    main("--full" in sys.argv)
