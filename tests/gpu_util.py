"""Helpers for the -m gpu parity tests: run the CUDA path through the C-ABI binding and compare with the oracle."""
from __future__ import annotations

import numpy as np


def gpu_run(w, K=4, max_neigh=None, stats=False, export=False, retry=False, hint=None, variant=None):
    """Build + traverse workload `w` on cuda:0.  Returns dict(nlist, n_neigh, M, [exports], [stats])."""
    import torch
    from paper_1901_08088_b200 import qbvh

    dev = torch.device("cuda:0")
    max_neigh = w.max_neigh if max_neigh is None else max_neigh
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, K)
    qbvh.qbvh_set_option(qbvh.OPT_STATS, int(stats))
    qbvh.qbvh_set_collapse_hint(hint)
    prev_variant = qbvh.qbvh_get_option(qbvh.OPT_VARIANT)
    if variant is not None:
        qbvh.qbvh_set_option(qbvh.OPT_VARIANT, variant)
    nl = qbvh.NeighborList(w.N, T=w.T, max_neigh=max_neigh, device=dev)
    pos = torch.from_numpy(w.pos).to(dev)
    typ = None if w.type is None else torch.from_numpy(w.type).to(dev)
    nl.build(pos, typ, w.box)
    out = {}
    if export:
        out["keys_sorted"] = qbvh.qbvh_debug_export(qbvh.EXPORT_KEYS_SORTED, w.N)
        out["perm"] = qbvh.qbvh_debug_export(qbvh.EXPORT_PERM, w.N)
        out["nodes"] = qbvh.qbvh_debug_export(qbvh.EXPORT_NODES, w.N)
        out["parent"] = qbvh.qbvh_debug_export(qbvh.EXPORT_PARENT, w.N)
        out["frames"] = qbvh.qbvh_debug_export(qbvh.EXPORT_FRAMES, w.N)
        out["segments"] = qbvh.qbvh_debug_export(qbvh.EXPORT_SEGMENTS, w.N)
        out["sorted_pos"] = qbvh.qbvh_debug_export(qbvh.EXPORT_SORTED_POS, w.N)
        out["counts"] = qbvh.qbvh_debug_export(qbvh.EXPORT_COUNTS, w.N)    # nodes written, query groups, cells, cell level
        out["nodes_emitted"] = int(out["counts"][0])
    nl.n_neigh.fill_(-7)
    nl.nlist.fill_(-1)
    M = nl.neighbors(w.r_list, retry=retry)
    torch.cuda.synchronize()
    out["M"] = M
    out["max_neigh"] = nl.max_neigh
    out["nlist"] = nl.nlist.cpu().numpy()[: w.N]
    out["n_neigh"] = nl.n_neigh.cpu().numpy()[: w.N]
    out["retries"] = nl.retries
    if stats:
        out["stats"] = qbvh.qbvh_get_stats()
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
    qbvh.qbvh_set_collapse_hint(None)
    qbvh.qbvh_set_option(qbvh.OPT_VARIANT, prev_variant)
    return out


def compare_with_oracle(w, out, oracle_csr, allow_overflow=False):
    """O3 of SURVEY.md §8c: per-row sets after sorting; counts; M; no self, no duplicates, indices in range.
    Returns a report dict; asserts the north_star bar (and, stricter, zero mismatches: both sides evaluate the
    same fp32 predicate)."""
    row_ptr, nbr, band = oracle_csr
    N = w.N
    cap = out["max_neigh"]
    n_or = np.diff(row_ptr).astype(np.int64)
    n_gpu = out["n_neigh"].astype(np.int64)
    assert np.array_equal(n_gpu, n_or), f"n_neigh differs on {np.sum(n_gpu != n_or)} rows"
    assert out["M"] == (int(n_or.max()) if N else 0)
    if not allow_overflow:
        assert out["M"] <= cap
    nlist = out["nlist"].astype(np.int64)
    cols = np.arange(nlist.shape[1])[None, :]
    valid = cols < np.minimum(n_gpu, cap)[:, None]
    assert np.all((nlist[valid] >= 0) & (nlist[valid] < N)), "index out of range"
    assert not np.any(nlist[valid] == np.broadcast_to(np.arange(N)[:, None], nlist.shape)[valid]), "self in list"
    big = np.iinfo(np.int64).max
    g = np.where(valid, nlist, big)
    g.sort(axis=1)
    assert not np.any((g[:, 1:] == g[:, :-1]) & (g[:, 1:] != big)), "duplicate entries in a row"
    # oracle as padded matrix
    o = np.full_like(g, big)
    ri = np.repeat(np.arange(N), n_or)
    ci = np.arange(len(nbr)) - np.repeat(row_ptr[:-1], n_or)
    keep = ci < nlist.shape[1]
    o[ri[keep], ci[keep]] = nbr[keep]
    full = n_or <= cap
    mism_rows = np.nonzero(np.any(g[full] != o[full], axis=1))[0]
    report = {"pairs": int(len(nbr)), "rows_checked": int(full.sum()), "rows_mismatched": int(len(mism_rows)),
              "in_band_pairs": int(band.sum()) if band is not None else None}
    only_gpu = only_or = oob = 0
    if len(mism_rows):
        fr = np.nonzero(full)[0]
        for r in fr[mism_rows][:1000]:
            a = set(g[r][g[r] != big].tolist())
            b = nbr[row_ptr[r]:row_ptr[r + 1]]
            bset = set(b.tolist())
            only_gpu += len(a - bset)
            only_or += len(bset - a)
            # out-of-band: oracle-only pairs whose band flag is 0 (gpu-only pairs cannot be classified here)
            bb = band[row_ptr[r]:row_ptr[r + 1]]
            oob += sum(1 for j, f in zip(b.tolist(), bb.tolist()) if j not in a and not f)
    report.update(only_gpu=only_gpu, only_oracle=only_or, out_of_band=oob)
    assert oob == 0, report
    assert (only_gpu + only_or) <= 1e-6 * max(len(nbr), 1), report
    assert len(mism_rows) == 0, report   # stricter than the bar: identical arithmetic => identical sets
    if allow_overflow:
        # rows over capacity hold `cap` distinct TRUE neighbors
        over = np.nonzero(~full)[0]
        for r in over[:2000]:
            a = g[r][:cap]
            assert len(np.unique(a)) == cap and np.all(np.isin(a, nbr[row_ptr[r]:row_ptr[r + 1]]))
        report["rows_overflowed"] = int(len(over))
    return report
