"""-m gpu parity tests: the CUDA path, called through the C-ABI binding, against the CPU oracle.

Bar (BASELINE.json north_star): bit-exact integer work (keys, permutation, node words, links); neighbor sets
identical after sorting except pairs within 1e-5 sigma of r_list (counted; <= 1e-6 of all pairs) — here both sides
evaluate the same fp32 predicate, so the tests additionally assert ZERO mismatches.
"""
import numpy as np
import pytest

from oracle import neighbors as ON
from oracle import tree as OT
from paper_1901_08088_b200 import workloads as W

from gpu_util import compare_with_oracle, gpu_run

pytestmark = pytest.mark.gpu


C_NODE, C_LEAF_FIXED, C_LEAF_PER_PARTICLE = 1, 16, 1   # DESIGN.md §3.7 (restated here, not imported)


def collapse_frontier(t, K, r_hint=None):
    """Subtree collapse restated on the oracle's one-particle-per-leaf tree.

    Bottom up: a single particle is 'pending'; an internal node with cnt <= K particles whose children are both
    pending collapses into one range leaf — always without a hint; with a hint r_b for its tree only if that does
    not raise the cost  W(n) (C_F + C_L cnt)  <=  W(n) C_N + sum over the two children of W(c) (C_F + C_L cnt_c),
    W = prod_d (max(q_hi,d - q_lo,d, 0) + 2 ceil(r_b / Delta_d)) in integers (bins of the tree's frame).
    Returns (emitted, collapsed): which nodes exist in the collapsed tree, which of them are range leaves."""
    N = t.N
    M = 2 * N - 1
    size = np.where(t.first >= 0, t.last - t.first + 1, 0).astype(np.int64)
    pend = np.zeros(M, bool)
    pend[N - 1:] = True
    coll = np.zeros(M, bool)
    ql = np.stack([(t.wlo >> (10 * d)) & 1023 for d in range(3)], 1).astype(np.int64)
    qh = np.stack([(t.whi >> (10 * d)) & 1023 for d in range(3)], 1).astype(np.int64)
    ext = np.maximum(qh - ql, 0)
    tree_of = np.searchsorted(t.seg[1:], np.maximum(t.first, 0), side="right")
    rb = None
    if r_hint is not None:
        rb = np.full((t.T, 3), -1, np.int64)
        for tb in range(t.T):
            if r_hint[tb] > 0 and t.roots[tb] >= 0:
                for d in range(3):
                    delta = np.float32(t.frames[tb, 6 + d])
                    rb[tb, d] = min(int(np.ceil(np.float32(r_hint[tb]) / delta)), 1023) if delta > 0 else 1

    def Wv(n):                                     # swollen-volume weight of nodes n (int64 array)
        r = rb[tree_of[n]]
        return (ext[n, 0] + 2 * r[:, 0]) * (ext[n, 1] + 2 * r[:, 1]) * (ext[n, 2] + 2 * r[:, 2])

    def leaf_cost(m):
        return Wv(m) * (C_LEAF_FIXED + C_LEAF_PER_PARTICLE * size[m])

    if K > 1:
        internal = np.arange(M) < N - 1
        for s in range(2, K + 1):                  # children (fewer particles) before parents; one size class at a time
            n = np.nonzero(internal & (size == s))[0]
            if len(n) == 0:
                continue
            a, b = t.left[n], t.right[n]
            ok = pend[a] & pend[b]
            if rb is not None:
                hinted = rb[tree_of[n], 0] >= 0
                cheaper = leaf_cost(n) <= Wv(n) * C_NODE + leaf_cost(a) + leaf_cost(b)
                ok &= np.where(hinted, cheaper, True)
            pend[n] = coll[n] = ok
    # top down, level by level: a node exists iff no proper ancestor collapsed
    emitted = np.zeros(M, bool)
    frontier = np.array([int(r) for r in t.roots if r >= 0], np.int64)
    while len(frontier):
        emitted[frontier] = True
        inner = frontier[(frontier < N - 1) & ~coll[frontier]]
        frontier = np.concatenate([t.left[inner], t.right[inner]]).astype(np.int64)
    return emitted, coll


def expected_nodes(t, K, r_hint=None):
    """Oracle tree -> (node array, emitted mask) the CUDA path must produce for collapse cap K and hint r_hint."""
    nodes = t.nodes_int4().copy()
    emitted, coll = collapse_frontier(t, K, r_hint)
    nodes[coll, 2] = ~t.first[coll]          # a range leaf: ~first; its particle count follows from its rope
    return nodes, emitted


def check_build(w, K, r_hint=None):
    out = gpu_run(w, K=K, export=True, hint=r_hint)
    t = OT.build(w.pos, w.type, w.box, T=w.T)
    N = w.N
    assert np.array_equal(out["keys_sorted"], t.key_sorted)                      # a1 + a2 keys
    assert np.array_equal(out["perm"].astype(np.int64), t.perm)                  # a2 stable permutation
    seg, roots = out["segments"][:5], out["segments"][5:9]
    assert np.array_equal(seg[: w.T + 1], t.seg) and np.all(seg[w.T:] == N)
    assert np.array_equal(roots[: w.T], t.roots) and np.all(roots[w.T:] == -1)
    for tb in range(w.T):
        if t.roots[tb] >= 0:
            assert np.array_equal(out["frames"][tb, :9], t.frames[tb])           # root boxes + Delta (bitwise)
    assert np.array_equal(out["sorted_pos"][:, :3], t.pos_sorted)               # a2' gather
    assert np.array_equal(out["sorted_pos"][:, 3].view(np.uint32).astype(np.int64), t.perm)
    exp, emitted = expected_nodes(t, K, r_hint)
    if K == 1:
        assert emitted.sum() == 2 * N - 1 - max(0, np.count_nonzero(np.diff(t.seg) > 0) - 1)   # the paper's tree, whole
    assert np.array_equal(out["nodes"][emitted], exp[emitted])                   # a3..a6: 16-byte nodes, bitwise
    assert np.array_equal(out["parent"][emitted], t.parent[emitted])
    assert out["nodes_emitted"] == int(emitted.sum())                            # descendants of range leaves are never written
    return out, t


@pytest.mark.parametrize("K", [1, 4, 16])
@pytest.mark.parametrize("cid", [1, 2, 3, 4, 5])
def test_build_parity_small(cid, K):
    check_build(W.make_config(cid, small=True), K)


@pytest.mark.parametrize("cid,K,hinted", [(2, 1, False), (2, 32, False), (2, 32, True), (3, 1, False), (3, 32, False),
                                          (5, 1, False), (5, 32, False)])
def test_build_parity_full_size(cid, K, hinted):
    """The build the benchmark times, bit for bit against the oracle tree (steps a1..a6 + the collapse): BASELINE.json
    sizes reach what the small cases cannot — Morton-cell levels 5 (configs 2, 3) and 6 (config 5), at level 6 the
    128-tile scan with its grid-wide meeting point, and at K = 32 the top-down split of the nodes above the range
    leaves (taken once N >= 32 x the resident warps of the traversal)."""
    w = W.make_config(cid)
    hint = np.asarray(w.r_list, np.float32).reshape(w.T, w.T).max(axis=0) if hinted else None
    out, t = check_build(w, K, r_hint=hint)
    assert int(out["counts"][3]) == (6 if cid == 5 else 5)


@pytest.mark.parametrize("N", [1, 2, 3, 31, 32, 33, 255, 4095, 4096, 4097, 8193, 70001])
def test_build_sizes_and_ragged_tiles(N):
    """Sort tiles are 4096 keys: sizes around the tile edge, one warp, one element."""
    w = W.lj_uniform(N=N, rho=min(0.85, N / 64.0), r_list=1.2, config_id=40)   # L >= 4 > 2 r_list
    out, t = check_build(w, 1)
    compare_with_oracle(w, out, ON.neighbor_list(w.pos, None, w.box, w.r_list))


def _line(N, reverse=False, dup=1):
    """Particles on the body diagonal -> strictly increasing Morton keys (already sorted / reversed / duplicated)."""
    L = 64.0
    t = (np.arange(N) // dup) / max(1, (N - 1) // dup + 1)
    p = np.repeat(t[:, None], 3, 1) * L
    if reverse:
        p = p[::-1]
    return W._finish(np.ascontiguousarray(p), L)


@pytest.mark.parametrize("case", ["sorted", "reverse", "dups", "all_equal"])
def test_sort_degenerate_orders(case):
    N = 20000
    if case == "all_equal":
        pos, box = W._finish(np.full((N, 3), 3.25), 64.0)
    else:
        pos, box = _line(N, reverse=(case == "reverse"), dup=(7 if case == "dups" else 1))
    w = W.Workload(case, pos, None, box, np.array([[0.5]], np.float32), 64)
    out, t = check_build(w, 4)
    if case == "all_equal":
        assert np.array_equal(out["perm"], np.arange(N))   # stability: equal keys keep input order


@pytest.mark.parametrize("K", [1, 4, 8, 16, 32])
@pytest.mark.parametrize("cid", [1, 2, 3, 4, 5])
def test_neighbors_parity_small(cid, K):
    w = W.make_config(cid, small=True)
    out = gpu_run(w, K=K)
    rep = compare_with_oracle(w, out, ON.neighbor_list(w.pos, w.type, w.box, w.r_list))
    assert rep["rows_checked"] == w.N


@pytest.mark.parametrize("cid", [2, 3, 4, 5])
def test_neighbors_parity_full_size(cid):
    """BASELINE.json's full sizes, in the launch configuration bench.py times (default options)."""
    w = W.make_config(cid)
    out = gpu_run(w, K=32)
    rep = compare_with_oracle(w, out, ON.neighbor_list(w.pos, w.type, w.box, w.r_list, method="cell"))
    assert rep["rows_checked"] == w.N and rep["pairs"] > 0


def test_overflow_detection_and_retry():
    w = W.lj_uniform()
    csr = ON.neighbor_list(w.pos, None, w.box, w.r_list)
    true_max = int(np.diff(csr[0]).max())
    out = gpu_run(w, max_neigh=64)                     # too small: mean count is ~87
    assert out["M"] == true_max > 64
    compare_with_oracle(w, out, csr, allow_overflow=True)
    out = gpu_run(w, max_neigh=64, retry=True)         # wrapper re-allocates with capacity >= M and calls again
    assert out["retries"] == 1 and out["max_neigh"] >= true_max
    compare_with_oracle(w, out, csr)
    out = gpu_run(w, max_neigh=0)                      # count-only use
    assert np.array_equal(out["n_neigh"], np.diff(csr[0]))


def test_edge_cases():
    import torch
    from paper_1901_08088_b200 import qbvh
    box = np.array([-5, -5, -5, 10, 10, 10], np.float32)
    # N = 0
    nl = qbvh.NeighborList(0, 1, 8)
    nl.build(torch.zeros((0, 3), device="cuda"), None, box)
    assert nl.neighbors(np.array([[1.0]], np.float32)) == 0
    # N = 1: the tree is one leaf that is also the root
    w = W.Workload("one", np.array([[1, 2, 3]], np.float32), None, box, np.array([[2.0]], np.float32), 4)
    out = gpu_run(w, export=True)
    assert out["M"] == 0 and out["n_neigh"].tolist() == [0] and out["segments"][5] == 0
    # two coincident particles are neighbors of each other; self excluded by index
    w = W.Workload("two", np.array([[1, 2, 3], [1, 2, 3]], np.float32), None, box, np.array([[0.1]], np.float32), 4)
    out = gpu_run(w)
    assert out["n_neigh"].tolist() == [1, 1] and out["nlist"][0, 0] == 1 and out["nlist"][1, 0] == 0
    # all particles share one coordinate (zero root extent along x) and faces
    rng = np.random.default_rng(5)
    p = rng.random((3000, 3)) * 10
    p[:, 0] = 2.5
    p[:40, 1] = 0.0
    pos, _ = W._finish(p, 10.0)
    w = W.Workload("plane", pos, None, box, np.array([[1.1]], np.float32), 256)
    for K in (1, 4):
        compare_with_oracle(w, gpu_run(w, K=K), ON.neighbor_list(w.pos, None, box, w.r_list))
    # four types, one of them empty, one with a single particle, one pair type switched off
    p = rng.random((5000, 3)) * 10
    pos, _ = W._finish(p, 10.0)
    typ = rng.integers(0, 2, 5000).astype(np.int32) * 2        # types 0 and 2
    typ[17] = 3
    r = np.array([[1.0, 0.5, 1.4, 2.0], [0.5, 0.5, 0.5, 0.5], [1.4, 0.5, 0.0, 3.0], [2.0, 0.5, 3.0, 1.0]], np.float32)
    w = W.Workload("types", pos, typ, box, r, 512)
    for K in (1, 4):
        compare_with_oracle(w, gpu_run(w, K=K), ON.neighbor_list(w.pos, typ, box, r))
    # r just under L/2 (padded radius still below L/2)
    w = W.Workload("halfbox", pos[:600], None, box, np.array([[4.99]], np.float32), 600)
    compare_with_oracle(w, gpu_run(w, K=4), ON.neighbor_list(w.pos, None, box, w.r_list))


def test_error_codes():
    import torch
    from paper_1901_08088_b200 import qbvh
    w = W.lj_uniform(N=1000, config_id=41)
    nl = qbvh.NeighborList(w.N, 1, 64)
    pos = torch.from_numpy(w.pos).cuda()
    nl.build(pos, None, w.box)
    with pytest.raises(qbvh.QbvhError) as e:
        nl.neighbors(np.array([[0.5 * float(w.box[3])]], np.float32))
    assert e.value.code == qbvh.ERR_CUTOFF_TOO_LARGE
    typ = torch.zeros(w.N, dtype=torch.int32, device="cuda")
    typ[5] = 3
    nl2 = qbvh.NeighborList(w.N, 2, 64)
    nl2.build(pos, typ, w.box)
    with pytest.raises(qbvh.QbvhError) as e:
        nl2.neighbors(np.ones((2, 2), np.float32))
    assert e.value.code == qbvh.ERR_TYPE_RANGE
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    qbvh.qbvh_set_workspace(small)
    with pytest.raises(qbvh.QbvhError) as e:
        qbvh.qbvh_build(pos, None, w.N, w.box)
    assert e.value.code == qbvh.ERR_WORKSPACE


def test_determinism_and_rebuild():
    w = W.make_config(2, small=True)
    a = gpu_run(w, K=4, export=True)
    b = gpu_run(w, K=4, export=True)
    assert np.array_equal(a["nodes"], b["nodes"]) and np.array_equal(a["perm"], b["perm"])
    assert np.array_equal(a["n_neigh"], b["n_neigh"])
    valid = np.arange(a["nlist"].shape[1])[None, :] < a["n_neigh"][:, None]     # entries past the count are unspecified
    assert np.array_equal(np.sort(np.where(valid, a["nlist"], 1 << 30), 1),
                          np.sort(np.where(valid, b["nlist"], 1 << 30), 1))


@pytest.mark.parametrize("cid", [1, 3, 5])
def test_census_matches_algorithm1_replay(cid):
    """K = 1 is the paper's tree; the instrumented traversal must take exactly the oracle's decisions:
    same number of node tests, leaf-box overlaps and overlapping images (PAPER.md:198 census)."""
    w = W.make_config(cid, small=True)
    out = gpu_run(w, K=1, stats=True)
    t = OT.build(w.pos, w.type, w.box, T=w.T)
    tr = OT.traverse(t, w.box, w.r_list)
    s = out["stats"]
    assert s["node_tests"] == int(tr["n_tests"].sum())
    assert s["leaf_overlaps"] == int(tr["n_overlap"].sum()) == s["dist_checks"]
    assert s["images"] == int(tr["n_images"].sum())
    assert s["neighbors"] == int(out["n_neigh"].sum())


@pytest.mark.parametrize("rho,key", [(0.2, "false_pos_per_particle_rho0.2"), (0.8, "false_pos_per_particle_rho0.8")])
def test_false_positive_census_vs_paper(rho, key):
    """1.5 / 3.8 false-positive neighbors per particle (N=128,000, r_c=3.0) — measured on the GPU."""
    from conftest import read_golden
    paper = {k: float(v) for k, v, _ in read_golden("paper_constants.txt")}[key]
    w = W.lj_uniform(N=128_000, rho=rho, r_list=3.0, config_id=100, max_neigh=160)
    out = gpu_run(w, K=1, stats=True)
    s = out["stats"]
    fp = (s["leaf_overlaps"] - w.N - s["neighbors"]) / w.N
    assert abs(fp - paper) / paper < 0.12, (fp, paper)


@pytest.mark.parametrize("pinned", [True, False])
def test_host_buffer_api_matches_device_api(pinned):
    """qbvh_build_host / qbvh_neighbors_host: pinned rows are written by the SMs (only the entries that exist),
    pageable rows by the copy engine; both give the device call's counts and the oracle's lists, and neither writes
    outside the rows (a guard band of the host buffer keeps its fill)."""
    import torch
    from paper_1901_08088_b200 import qbvh
    w = W.make_config(3, small=True)
    dev_out = gpu_run(w, K=4)
    qbvh.qbvh_set_num_types(w.T)
    ws = torch.empty(qbvh.qbvh_workspace_bytes(w.N, w.T), dtype=torch.uint8, device="cuda")
    stg = torch.empty(qbvh.qbvh_staging_bytes(w.N, w.max_neigh), dtype=torch.uint8, device="cuda")
    qbvh.qbvh_set_workspace(ws)
    qbvh.qbvh_set_staging(stg)
    pos, typ = torch.from_numpy(w.pos), torch.from_numpy(w.type)
    guard = 64
    buf = torch.full(((w.N + 2 * guard) * w.max_neigh,), -9, dtype=torch.int32)
    n_neigh = torch.empty(w.N, dtype=torch.int32)
    if pinned:
        pos, typ, buf, n_neigh = pos.pin_memory(), typ.pin_memory(), buf.pin_memory(), n_neigh.pin_memory()
    nlist = buf[guard * w.max_neigh: (guard + w.N) * w.max_neigh].view(w.N, w.max_neigh)
    qbvh.qbvh_build_host(pos, typ, w.N, w.box)
    M = qbvh.qbvh_neighbors_host(w.r_list, nlist, n_neigh, w.max_neigh)
    assert M == dev_out["M"] and np.array_equal(n_neigh.numpy(), dev_out["n_neigh"])
    out = {"M": M, "max_neigh": w.max_neigh, "nlist": nlist.numpy(), "n_neigh": n_neigh.numpy()}
    compare_with_oracle(w, out, ON.neighbor_list(w.pos, w.type, w.box, w.r_list))
    b = buf.numpy()
    assert (b[: guard * w.max_neigh] == -9).all() and (b[(guard + w.N) * w.max_neigh:] == -9).all()
    cnt = n_neigh.numpy().astype(np.int64)
    if pinned:   # the bytes that crossed: counts + 16-byte pieces of the rows + two result words
        assert qbvh.qbvh_last_d2h_bytes() == 4 * w.N + 16 + int((16 * ((np.minimum(cnt, w.max_neigh) + 3) // 4)).sum())
        # nothing beyond the last 16-byte piece of a row was written
        i = int(np.argmin(cnt))
        assert (nlist.numpy()[i, 4 * ((cnt[i] + 3) // 4):] == -9).all()
    else:
        assert qbvh.qbvh_last_d2h_bytes() == 4 * w.N + 8 + 4 * min(M, w.max_neigh) * w.N
    qbvh.qbvh_set_staging(None)


@pytest.mark.parametrize("cid", [1, 3, 5])
def test_count_overlaps_is_the_papers_kernel(cid):
    """qbvh_count_overlaps = Algorithm 1 as printed (accept on leaf-box overlap) on the paper's
    one-particle-per-leaf tree: per particle the oracle replay's count, minus the particle's own leaf."""
    import torch
    from paper_1901_08088_b200 import qbvh
    w = W.make_config(cid, small=True)
    dev = torch.device("cuda:0")
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, 1)
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
    nl = qbvh.NeighborList(w.N, T=w.T, max_neigh=w.max_neigh, device=dev)   # owns the workspace: keep it alive
    nl.build(torch.from_numpy(w.pos).to(dev), None if w.type is None else torch.from_numpy(w.type).to(dev), w.box)
    t = OT.build(w.pos, w.type, w.box, T=w.T)
    tr = OT.traverse(t, w.box, w.r_list)
    cnt = torch.full((w.N,), -7, dtype=torch.int32, device=dev)
    M = qbvh.qbvh_count_overlaps(w.r_list, cnt)
    got = cnt.cpu().numpy()
    r = np.asarray(w.r_list, np.float32).reshape(w.T, w.T)
    ta = np.searchsorted(t.seg[1:], np.arange(w.N), side="right")        # type of sorted position k
    own = (r[ta, ta] > 0).astype(np.int64)                                # own leaf overlaps iff its own tree is walked
    expect = tr["n_overlap"].astype(np.int64) - own
    assert np.array_equal(got[t.perm], expect)
    assert M == int(expect.max())
    # and it brackets the exact list: every true neighbor's leaf box overlaps
    nl.neighbors(w.r_list)
    assert np.all(got >= nl.n_neigh.cpu().numpy()[: w.N])


@pytest.mark.parametrize("K", [1, 8])
@pytest.mark.parametrize("cid", [1, 3, 4])
def test_algorithm1_kernel_list_parity(cid, K):
    """QBVH_OPT_VARIANT = 0: Algorithm 1 as written (one thread per particle) with the exact leaf
    filter must emit the same lists as the oracle (and hence as the production kernel)."""
    from paper_1901_08088_b200 import qbvh
    w = W.make_config(cid, small=True)
    qbvh.qbvh_set_option(qbvh.OPT_VARIANT, 0)
    try:
        out = gpu_run(w, K=K)
    finally:
        qbvh.qbvh_set_option(qbvh.OPT_VARIANT, 1)
    rep = compare_with_oracle(w, out, ON.neighbor_list(w.pos, w.type, w.box, w.r_list))
    assert rep["rows_checked"] == w.N


def test_randomized_inputs_stress():
    """Seeded random systems: sizes around warp/tile edges, 1-4 types with empty and rare ones, clustered, flat and
    duplicated coordinates, skipped type pairs, odd row capacities (vector and scalar store paths, overflow), every
    collapse threshold.  Each list must equal the oracle's."""
    rng = np.random.default_rng(20240607)
    for it in range(60):
        N = int(rng.choice([1, 2, 5, 33, 100, 777, 3000, 9000]))
        T = int(rng.choice([1, 1, 2, 3, 4]))
        L = rng.uniform(6.0, 30.0, 3) * np.array([1, 1, rng.choice([1, 3])])
        pos = rng.random((N, 3)) * L
        if rng.random() < 0.5 and N > 10:
            c = rng.random((max(1, N // 50), 3)) * L
            pos[: N // 2] = (c[rng.integers(0, len(c), N // 2)] + rng.normal(0, 0.4, (N // 2, 3))) % L
        if rng.random() < 0.2:
            pos[:, 2] = L[2] * 0.25
        if rng.random() < 0.2 and N > 3:
            pos[1] = pos[0]
        typ = None
        if T > 1:
            typ = rng.choice(T, N, p=rng.dirichlet(np.ones(T) * 0.5)).astype(np.int32)
        p32, box = W._finish(pos, L)
        r = rng.uniform(0.5, min(0.45 * float(L.min()), 4.0), (T, T)).astype(np.float32)
        r = np.maximum(r, r.T)
        if T > 1 and rng.random() < 0.3:
            r[0, 1] = r[1, 0] = 0.0
        cap = int(rng.choice([0, 3, 4, 12, 16, 50, 64, 200]))
        K = int(rng.choice([1, 2, 4, 8, 16, 32]))
        w = W.Workload(f"stress{it}", p32, typ, box, r, cap)
        out = gpu_run(w, K=K, max_neigh=cap)
        csr = ON.neighbor_list(w.pos, w.type, w.box, w.r_list, method="brute" if N <= 3000 else "cell")
        compare_with_oracle(w, out, csr, allow_overflow=True)


# ---------------------------------------------------------------------------------------------------------------
# Round-2 additions: boxes whose origin is not -L/2, the boundary pairs of the pad pin, Algorithm 1 as printed at
# BASELINE sizes, the work-list bound, rebuilding in place on one workspace.
# ---------------------------------------------------------------------------------------------------------------
ORIGINS = [(0.0, 0.0, 0.0), (1000.0, -3000.0, 17.0), (65536.0, -65536.0, 32768.0)]


@pytest.mark.parametrize("lo", ORIGINS)
@pytest.mark.parametrize("cid", [1, 3, 5])
def test_noncentred_box(cid, lo):
    """box_lo enters the Morton binning (a1), the entry-cell selection and the pad: keys, nodes and lists must match
    the oracle in boxes that do not start at -L/2 (far from the origin the fp32 grid is coarse: 2^-7 at 65536)."""
    w = W.shifted(W.make_config(cid, small=True), lo)
    for K in (1, 32):
        out, t = check_build(w, K)
        rep = compare_with_oracle(w, out, ON.neighbor_list(w.pos, w.type, w.box, w.r_list))
        assert rep["rows_checked"] == w.N


@pytest.mark.parametrize("lo", ORIGINS + [(-12.0, -12.0, -12.0)])
def test_boundary_pairs_across_faces_and_corners(lo):
    """The inputs of tests/test_oracle_tree.py::test_boundary_pairs_...: pairs at exactly r, one grid step inside and
    outside, through face and corner images.  Production kernel and Algorithm 1 as printed, K = 1 and collapsed."""
    from adversarial_inputs import boundary_pairs
    from paper_1901_08088_b200 import qbvh
    L, r, grid = 24.0, 3.0, 2.0 ** -6
    p, lo64 = boundary_pairs(lo, L, r, grid)
    pos, box = W.place(p, L, lo64)
    w = W.Workload("boundary", pos, None, box, np.array([[r]], np.float32), 128)
    csr = ON.neighbor_list(w.pos, None, w.box, w.r_list, method="brute")
    for variant in (1, 0):
        qbvh.qbvh_set_option(qbvh.OPT_VARIANT, variant)
        try:
            for K in (1, 8, 32):
                compare_with_oracle(w, gpu_run(w, K=K), csr)
        finally:
            qbvh.qbvh_set_option(qbvh.OPT_VARIANT, 1)


@pytest.mark.parametrize("cid", [2, 5])
def test_algorithm1_as_printed_full_size(cid):
    """BASELINE sizes through the paper's own kernels: variant 0 (Algorithm 1, one thread per particle, exact leaf
    filter) must emit the oracle's lists, and qbvh_count_overlaps on the one-particle-per-leaf tree must equal the
    CPU replay of Algorithm 1 per particle."""
    import torch
    from paper_1901_08088_b200 import qbvh
    w = W.make_config(cid)
    qbvh.qbvh_set_option(qbvh.OPT_VARIANT, 0)
    try:
        out = gpu_run(w, K=1)
    finally:
        qbvh.qbvh_set_option(qbvh.OPT_VARIANT, 1)
    rep = compare_with_oracle(w, out, ON.neighbor_list(w.pos, w.type, w.box, w.r_list, method="cell"))
    assert rep["rows_checked"] == w.N
    dev = torch.device("cuda:0")
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, 1)
    nl = qbvh.NeighborList(w.N, T=w.T, max_neigh=1, device=dev)
    nl.build(torch.from_numpy(w.pos).to(dev), None, w.box)
    cnt = torch.full((w.N,), -7, dtype=torch.int32, device=dev)
    M = qbvh.qbvh_count_overlaps(w.r_list, cnt)
    t = OT.build(w.pos, w.type, w.box, T=w.T)
    tr = OT.traverse(t, w.box, w.r_list)
    expect = tr["n_overlap"].astype(np.int64) - 1                       # minus the particle's own leaf
    assert np.array_equal(cnt.cpu().numpy()[t.perm], expect) and M == int(expect.max())
    assert np.all(expect[np.argsort(t.perm)] >= out["n_neigh"])        # brackets the exact list


def test_work_list_bound():
    """The warp work list of the production traversal: a cutoff that reaches everything in a dense,
    duplicate-ridden cloud drives the list to its 192-entry breadth-first fill and then into the one-entry depth-first
    mode over deep subtrees (duplicates extend the tree by the index bits).  Lists must still equal the oracle's and
    no bound may be reported violated (QBVH_ERR_INTERNAL would raise)."""
    rng = np.random.default_rng(77)
    L = 64.0
    base = rng.random((600, 3)) * 6.0 + 29.0                  # a blob in the middle of the box
    comb = 32.0 + 24.0 * 2.0 ** -np.arange(1, 25)[:, None] * np.ones((1, 3))   # a comb: keys with ever longer common prefixes
    p = np.concatenate([np.repeat(base, 8, axis=0), np.repeat(comb, 16, axis=0), rng.random((300, 3)) * L])
    p = p[rng.permutation(len(p))]
    pos, box = W._finish(p, L)
    for r, cap in ((30.0, 5600), (5.0, 5600)):
        w = W.Workload("worklist", pos, None, box, np.array([[r]], np.float32), cap)
        csr = ON.neighbor_list(w.pos, None, w.box, w.r_list, method="brute")
        for K in (1, 2, 32):
            compare_with_oracle(w, gpu_run(w, K=K), csr)


def test_rebuild_in_place_on_one_workspace():
    """What an MD code does: qbvh_build again and again on ONE workspace.  The meeting slots of the tree builder are
    not cleared between builds, stale ones are told apart by a per-build tag.  Same N, different
    positions / types / K each time, nodes, parents and lists compared with the oracle after every build, and the
    18-bit tag driven through its wrap."""
    TAG_MAX = (1 << 18) - 1
    import torch
    from paper_1901_08088_b200 import qbvh
    dev = torch.device("cuda:0")
    N, T = 30_000, 2
    rng = np.random.default_rng(11)
    nl = qbvh.NeighborList(N, T=T, max_neigh=256, device=dev)
    box_L = 40.0
    tags = []
    for it in range(7):
        p = rng.random((N, 3)) * box_L
        if it % 2:
            p[: N // 3] = (p[: N // 3] * 0.2 + 10.0)            # a dense clump: another tree shape on the same slots
        pos, box = W._finish(p, box_L)
        typ = (rng.random(N) < (0.1 + 0.1 * it)).astype(np.int32)
        r = np.array([[1.3, 1.1], [1.1, 0.9 + 0.05 * it]], np.float32)
        K = [1, 32, 4, 1, 16, 32, 2][it]
        qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, K)
        if it == 3:
            nl._activate()
            qbvh.qbvh_set_option(qbvh.OPT_DEBUG_BUILD_TAG, TAG_MAX - 1)   # this build: max - 1, next: max, then the wrap
        nl.build(torch.from_numpy(pos).to(dev), torch.from_numpy(typ).to(dev), box)
        tags.append(qbvh.qbvh_get_option(qbvh.OPT_DEBUG_BUILD_TAG))
        w = W.Workload(f"rebuild{it}", pos, typ, box, r, 256)
        t = OT.build(pos, typ, box, T=T)
        nodes = qbvh.qbvh_debug_export(qbvh.EXPORT_NODES, N)
        parent = qbvh.qbvh_debug_export(qbvh.EXPORT_PARENT, N)
        exp, emitted = expected_nodes(t, K)
        assert np.array_equal(nodes[emitted], exp[emitted]), it
        assert np.array_equal(parent[emitted], t.parent[emitted]), it
        nl.n_neigh.fill_(-7)
        M = nl.neighbors(r, retry=False)
        out = {"M": M, "max_neigh": nl.max_neigh, "nlist": nl.nlist.cpu().numpy()[:N], "n_neigh": nl.n_neigh.cpu().numpy()[:N]}
        compare_with_oracle(w, out, ON.neighbor_list(pos, typ, box, r))
    assert tags == [1, 2, 3, TAG_MAX - 1, TAG_MAX, 1, 2], tags    # no clearing between builds except at the wrap
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, 32)


@pytest.mark.parametrize("K", [8, 32])
@pytest.mark.parametrize("cid", [1, 2, 3, 4, 5])
def test_collapse_heuristic_build_and_lists(cid, K):
    """build-side subtree collapse chosen by the cost heuristic (qbvh_set_collapse_hint).  The node
    array must hold exactly the nodes at or above the frontier the heuristic picks on the oracle's
    one-particle-per-leaf tree (restated in collapse_frontier above), bit for bit, and nothing below it; lists stay
    identical to the oracle's."""
    w = W.make_config(cid, small=True)
    hint = np.asarray(w.r_list, np.float32).reshape(w.T, w.T).max(axis=0)
    out, t = check_build(w, K, r_hint=hint)
    rep = compare_with_oracle(w, out, ON.neighbor_list(w.pos, w.type, w.box, w.r_list))
    assert rep["rows_checked"] == w.N
    emitted, coll = collapse_frontier(t, K, hint)
    # the heuristic is not the plain size threshold: on a type far sparser than its cutoff it stops earlier
    plain, _ = collapse_frontier(t, K, None)
    assert emitted.sum() >= plain.sum()
    if cid == 3 and K == 32:
        assert emitted.sum() > plain.sum()


# ---------------------------------------------------------------------------------------------------------------
# double-precision particle data (fp32 tree, padded fp32 search, fp64 leaf predicate)
# ---------------------------------------------------------------------------------------------------------------
def gpu_run_f64(pos64, typ, box64, r64, T, max_neigh, K=32):
    import torch
    from paper_1901_08088_b200 import qbvh
    dev = torch.device("cuda:0")
    N = len(pos64)
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, K)
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
    qbvh.qbvh_set_collapse_hint(None)
    nl = qbvh.NeighborList(N, T=T, max_neigh=max_neigh, device=dev)
    nl.build(torch.from_numpy(pos64).to(dev), None if typ is None else torch.from_numpy(typ).to(dev), box64)
    nl.n_neigh.fill_(-7)
    nl.nlist.fill_(-1)
    M = nl.neighbors(r64, retry=False)
    torch.cuda.synchronize()
    out = {"M": M, "max_neigh": nl.max_neigh, "nlist": nl.nlist.cpu().numpy()[:N], "n_neigh": nl.n_neigh.cpu().numpy()[:N]}
    out["keys_sorted"] = qbvh.qbvh_debug_export(qbvh.EXPORT_KEYS_SORTED, N)
    out["nodes"] = qbvh.qbvh_debug_export(qbvh.EXPORT_NODES, N)
    out["perm"] = qbvh.qbvh_debug_export(qbvh.EXPORT_PERM, N)
    return out


@pytest.mark.parametrize("K", [1, 32])
@pytest.mark.parametrize("cid", [1, 2, 3, 4, 5])
def test_f64_particles_parity_small(cid, K):
    """qbvh_build_f64 / qbvh_neighbors_f64 against the fp64 oracle: identical sets, zero mismatches (both sides evaluate
    the same fp64 predicate; the fp32 stage only prunes).  The tree must be the fp32 tree of the rounded positions."""
    w = W.make_config(cid, small=True)
    pos64, box64, r64 = W.as_f64(w)
    out = gpu_run_f64(pos64, w.type, box64, r64, w.T, w.max_neigh, K=K)
    w64 = W.Workload(w.name + "_f64", w.pos, w.type, w.box, w.r_list, w.max_neigh)
    rp, nb = ON.neighbor_list_f64(pos64, w.type, box64, r64)
    compare_with_oracle(w64, out, (rp, nb, np.zeros(len(nb), np.uint8)))
    t = OT.build(pos64.astype(np.float32), w.type, box64.astype(np.float32), T=w.T)     # the fp32 tree of the rounded positions
    exp, emitted = expected_nodes(t, K)
    assert np.array_equal(out["keys_sorted"], t.key_sorted) and np.array_equal(out["perm"].astype(np.int64), t.perm)
    assert np.array_equal(out["nodes"][emitted], exp[emitted])


def test_f64_resolves_what_fp32_cannot():
    """Pairs placed r (1 -+ 1e-10) apart at coordinates near 1000 (where fp32 resolves 6e-5): the fp64 path must accept
    the inner and reject the outer ones; through faces and a corner as well."""
    rng = np.random.default_rng(3)
    r = 2.5
    lo = np.array([990.0, -5.0, 300.0])
    L = np.array([40.0, 40.0, 40.0])
    box64 = np.concatenate([lo, L])
    base = lo + np.array([[0.3, 0.3, 0.3], [20.0, 0.2, 39.9], [39.8, 39.7, 39.9], [7.0, 21.0, 33.0]])
    pts, expect_pairs = [], []
    for b in base:
        i = len(pts)
        pts.append(b)
        for sgn in (+1, -1):
            for eps, inside in ((-1e-10, True), (+1e-10, False), (-3e-6, True), (+3e-6, False)):
                u = rng.normal(size=3)
                u /= np.linalg.norm(u)
                q = b + sgn * r * (1 + eps) * u
                q = lo + np.mod(q - lo, L)
                pts.append(q)
                if inside:
                    expect_pairs.append((i, len(pts) - 1))
    pos64 = np.array(pts)
    r64 = np.array([[r]])
    out = gpu_run_f64(pos64, None, box64, r64, 1, 32, K=4)
    rp, nb = ON.neighbor_list_f64(pos64, None, box64, r64, method="brute")
    w = W.Workload("f64pairs", pos64.astype(np.float32), None, box64.astype(np.float32), r64.astype(np.float32), 32)
    compare_with_oracle(w, out, (rp, nb, np.zeros(len(nb), np.uint8)))
    for i, j in expect_pairs:
        assert j in out["nlist"][i, : out["n_neigh"][i]]
    assert len(nb) >= 2 * len(expect_pairs)


def test_f64_full_size_config2():
    w = W.make_config(2)
    pos64, box64, r64 = W.as_f64(w)
    out = gpu_run_f64(pos64, None, box64, r64, 1, w.max_neigh, K=32)
    rp, nb = ON.neighbor_list_f64(pos64, None, box64, r64, method="cell")
    rep = compare_with_oracle(w, out, (rp, nb, np.zeros(len(nb), np.uint8)))
    assert rep["rows_checked"] == w.N


# ---------------------------------------------------------------------------------------------------------------
# query sharding.  One GPU here, so the ranks' calls are made one after another on one tree:
# qbvh_neighbors_range for every Z-order slice, merged, must be the oracle's list.
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("world", [2, 3, 7])
@pytest.mark.parametrize("cid", [1, 3, 5])
def test_query_sharding_slices_merge_to_the_oracle(cid, world):
    import torch
    from paper_1901_08088_b200 import qbvh, sharded
    w = W.make_config(cid, small=True)
    dev = torch.device("cuda:0")
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, 32)
    qbvh.qbvh_set_collapse_hint(None)
    be = sharded.CudaBackend(w.N, w.T, 16, dev)                    # capacity too small on purpose: the retry path
    be.build(torch.from_numpy(w.pos).to(dev), None if w.type is None else torch.from_numpy(w.type).to(dev), w.box)
    parts = []
    for g in range(world):
        first, count = sharded.slice_bounds(w.N, world, g)
        rows, n_neigh, nlist, M = be.neighbors_range(w.r_list, first, count)
        parts.append((rows.cpu().numpy(), n_neigh.cpu().numpy(), nlist.cpu().numpy()))
        assert M == (int(n_neigh.max().item()) if count else 0)
    n_all, l_all = sharded.merge_slices(w.N, parts)
    out = {"M": int(n_all.max()), "max_neigh": l_all.shape[1], "nlist": l_all, "n_neigh": n_all}
    compare_with_oracle(w, out, ON.neighbor_list(w.pos, w.type, w.box, w.r_list))
    # world size 1 through the distributed wrapper (no process group: a single rank)
    snl = sharded.ShardedNeighborList(w.N, T=w.T, max_neigh=w.max_neigh, device=dev)
    snl.build(torch.from_numpy(w.pos).to(dev), None if w.type is None else torch.from_numpy(w.type).to(dev), w.box)
    rows, n_neigh, nlist, M = snl.neighbors(w.r_list)
    n1, l1 = sharded.merge_slices(w.N, [(rows.cpu().numpy(), n_neigh.cpu().numpy(), nlist.cpu().numpy())])
    assert np.array_equal(n1, n_all)


@pytest.mark.parametrize("K,hinted", [(8, False), (1, False), (32, True)])
def test_query_sharding_on_other_builds(K, hinted):
    """qbvh_neighbors_range on trees other than the default K = 32 one: smaller range leaves (other tile widths of the
    traversal), the paper's one-particle leaves, and a build with the collapse hint."""
    import torch
    from paper_1901_08088_b200 import qbvh, sharded
    w = W.make_config(3, small=True)
    dev = torch.device("cuda:0")
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, K)
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
    qbvh.qbvh_set_collapse_hint(np.asarray(w.r_list, np.float32).reshape(w.T, w.T).max(axis=0) if hinted else None)
    try:
        be = sharded.CudaBackend(w.N, w.T, w.max_neigh, dev)
        be.build(torch.from_numpy(w.pos).to(dev), torch.from_numpy(w.type).to(dev), w.box)
        parts = []
        for g in range(3):
            first, count = sharded.slice_bounds(w.N, 3, g)
            rows, n_neigh, nlist, M = be.neighbors_range(w.r_list, first, count)
            parts.append((rows.cpu().numpy(), n_neigh.cpu().numpy(), nlist.cpu().numpy()))
    finally:
        qbvh.qbvh_set_collapse_hint(None)
        qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, 32)
    n_all, l_all = sharded.merge_slices(w.N, parts)
    out = {"M": int(n_all.max()), "max_neigh": l_all.shape[1], "nlist": l_all, "n_neigh": n_all}
    compare_with_oracle(w, out, ON.neighbor_list(w.pos, w.type, w.box, w.r_list))


@pytest.mark.parametrize("N,T,lvl", [(1, 1, 2), (3072, 1, 2), (3073, 1, 3), (200_000, 1, 5), (200_000, 4, 5), (1_600_000, 1, 6), (1_600_000, 2, 5)])
def test_cell_grid_level_choice(N, T, lvl):
    """The Morton-cell grid of the build: the smallest 2^lvl-per-axis grid with at most 48 particles per
    cell on average, lvl in [2, 6], T * 8^lvl <= 2^18 — and the build is correct on every side of those thresholds
    (counts against the oracle; the build products are compared bitwise in the other tests)."""
    rng = np.random.default_rng(N + T)
    L = max(4.0, (N / 0.85) ** (1 / 3))
    pos, box = W._finish(rng.random((N, 3)) * L, L)
    typ = None if T == 1 else rng.integers(0, T, N).astype(np.int32)
    r = np.full((T, T), 1.3, np.float32)
    w = W.Workload(f"lvl{N}_{T}", pos, typ, box, r, 40)
    out = gpu_run(w, K=32, export=True)
    assert int(out["counts"][3]) == lvl
    compare_with_oracle(w, out, ON.neighbor_list(pos, typ, box, r), allow_overflow=True)


def test_enqueue_result_is_qbvh_neighbors_in_two_halves():
    """qbvh_neighbors_enqueue + qbvh_neighbors_result: same lists, counts and M as qbvh_neighbors; a result without
    an enqueue, or after a rebuild, is refused."""
    import torch
    from paper_1901_08088_b200 import qbvh
    w = W.make_config(1)
    dev = torch.device("cuda:0")
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, 32)
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
    nl = qbvh.NeighborList(w.N, T=w.T, max_neigh=w.max_neigh, device=dev)
    nl.build(torch.from_numpy(w.pos).to(dev), None, w.box)
    M0 = nl.neighbors(w.r_list, retry=False)
    ref_cnt, ref_list = nl.n_neigh.clone(), nl.nlist.clone()
    nl.n_neigh.fill_(-1)
    nl.nlist.fill_(-1)
    nl.neighbors_enqueue(w.r_list)
    assert nl.neighbors_result() == M0
    assert torch.equal(nl.n_neigh, ref_cnt)
    a, b = nl.nlist.cpu().numpy(), ref_list.cpu().numpy()
    c = ref_cnt.cpu().numpy()
    for i in range(w.N):
        assert np.array_equal(np.sort(a[i, :c[i]]), np.sort(b[i, :c[i]]))
    with pytest.raises(qbvh.QbvhError):
        qbvh.qbvh_neighbors_result()                      # nothing enqueued any more
    nl.neighbors_enqueue(w.r_list)
    nl.build(torch.from_numpy(w.pos).to(dev), None, w.box)   # a rebuild drops the pending result
    with pytest.raises(qbvh.QbvhError):
        qbvh.qbvh_neighbors_result()
    torch.cuda.synchronize()
