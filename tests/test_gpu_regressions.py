"""-m gpu regression tests for findings of the round-2 review: argument combinations and call sequences
that the parity tests do not reach."""
import numpy as np
import pytest

from oracle import neighbors as ON
from paper_1901_08088_b200 import workloads as W

from gpu_util import compare_with_oracle

pytestmark = pytest.mark.gpu


def _built(w, max_neigh=None, K=32):
    import torch
    from paper_1901_08088_b200 import qbvh
    dev = torch.device("cuda:0")
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, K)
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
    qbvh.qbvh_set_option(qbvh.OPT_VARIANT, 1)
    qbvh.qbvh_set_collapse_hint(None)
    nl = qbvh.NeighborList(w.N, T=w.T, max_neigh=w.max_neigh if max_neigh is None else max_neigh, device=dev)
    nl.build(torch.from_numpy(w.pos).to(dev), None if w.type is None else torch.from_numpy(w.type).to(dev), w.box)
    return nl


def test_range_call_refuses_the_census_and_leaves_its_buffers_alone():
    """qbvh_neighbors_range hands the library buffers of `count` rows; the census of QBVH_OPT_STATS writes a row for
    every one of the N particles.  The combination is refused (INVALID_ARG) before anything is enqueued: guard bands
    around the slice's buffers stay intact.  With the option off again the same call works."""
    import torch
    from paper_1901_08088_b200 import qbvh
    w = W.make_config(1)
    nl = _built(w)
    first, count, cap, guard = 1000, 200, w.max_neigh, 4096
    lst = torch.full((guard + count * cap + guard,), -77, dtype=torch.int32, device=nl.device)
    cnt = torch.full((guard + count + guard,), -77, dtype=torch.int32, device=nl.device)
    try:
        qbvh.qbvh_set_option(qbvh.OPT_STATS, 1)
        with pytest.raises(qbvh.QbvhError) as e:
            qbvh.qbvh_neighbors_range(w.r_list, lst[guard:], cnt[guard:], cap, first, count)
        assert e.value.code == qbvh.ERR_INVALID_ARG
        torch.cuda.synchronize()
        assert torch.all(lst == -77) and torch.all(cnt == -77)
    finally:
        qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
    M = qbvh.qbvh_neighbors_range(w.r_list, lst[guard:], cnt[guard:], cap, first, count)
    torch.cuda.synchronize()
    assert torch.all(lst[:guard] == -77) and torch.all(lst[guard + count * cap:] == -77)
    assert torch.all(cnt[:guard] == -77) and torch.all(cnt[guard + count:] == -77)
    assert M == int(cnt[guard:guard + count].max().item()) > 0


def test_a_synchronous_call_drops_a_pending_enqueue():
    """After qbvh_neighbors_enqueue, any synchronous neighbor call overwrites the result words: a later
    qbvh_neighbors_result must say so (NOT_BUILT) instead of returning the other call's numbers."""
    import torch
    from paper_1901_08088_b200 import qbvh
    w = W.make_config(1)
    nl = _built(w)
    n_over = torch.zeros(w.N, dtype=torch.int32, device=nl.device)
    for sync_call in (lambda: nl.neighbors(w.r_list, retry=False),
                      lambda: qbvh.qbvh_count_overlaps(w.r_list, n_over),
                      lambda: qbvh.qbvh_neighbors_range(w.r_list, nl.nlist, nl.n_neigh, nl.max_neigh, 0, 10)):
        nl.neighbors_enqueue(w.r_list)
        sync_call()
        with pytest.raises(qbvh.QbvhError) as e:
            qbvh.qbvh_neighbors_result()
        assert e.value.code == qbvh.ERR_NOT_BUILT
    nl.neighbors_enqueue(w.r_list)                       # and the pair still works afterwards
    assert nl.neighbors_result() == nl.neighbors(w.r_list, retry=False)


def test_f64_box_that_is_not_representable_in_fp32():
    """qbvh_build_f64 with box64 != (double)(float)box64: origin and lengths that are not fp32 numbers, particles on
    the lower faces exactly and one ulp64 below the upper faces, partners across faces and a corner at r (1 -+ eps).
    Their fp32 roundings fall on or outside the rounded box; the lists must still be the fp64 definition's."""
    from test_gpu_parity import gpu_run_f64
    rng = np.random.default_rng(11)
    lo = np.array([0.1, -1.0 / 3.0, 1000.0 / 7.0])
    L = np.array([10.1, 9.7, 11.3])
    box64 = np.concatenate([lo, L])
    assert np.any(box64 != box64.astype(np.float32).astype(np.float64))
    hi_in = np.nextafter(lo + L, -np.inf)                          # the largest coordinates inside [lo, lo + L)
    r = 1.3
    pts = [lo.copy(), hi_in.copy()]
    for d in range(3):                                            # one coordinate on a face, the others inside
        for face in (lo[d], hi_in[d]):
            for _ in range(4):
                p = lo + rng.random(3) * L * 0.999
                p[d] = face
                pts.append(p)
    base = list(pts)
    for b in base:                                                # partners at r (1 -+ eps): across the face for most
        for eps in (-1e-9, 1e-9, -2e-6, 2e-6):
            u = rng.normal(size=3)
            u /= np.linalg.norm(u)
            q = b + r * (1 + eps) * u
            q = lo + np.mod(q - lo, L)
            pts.append(np.minimum(np.maximum(q, lo), hi_in))
    pts.extend(lo + rng.random((3000, 3)) * L)                    # a fluid around them
    pos64 = np.ascontiguousarray(np.array(pts))
    assert np.all(pos64 >= lo) and np.all(pos64 < lo + L)
    p32 = pos64.astype(np.float32)
    b32 = box64.astype(np.float32)
    assert np.any(p32 < b32[:3]) or np.any(p32 >= b32[:3] + b32[3:])     # the case the header allows and nothing covered
    r64 = np.array([[r]])
    for K in (1, 32):
        out = gpu_run_f64(pos64, None, box64, r64, 1, 64, K=K)
        rp, nb = ON.neighbor_list_f64(pos64, None, box64, r64, method="brute")
        w = W.Workload("f64box", p32, None, b32, r64.astype(np.float32), 64)
        rep = compare_with_oracle(w, out, (rp, nb, np.zeros(len(nb), np.uint8)))
        assert rep["rows_checked"] == len(pos64) and rep["pairs"] > 10000


def test_cell_scan_without_the_meeting_point():
    """The 128-tile scan of the build (cell grid level 6) lets its blocks meet once, with a bounded wait; a block that
    gives up sums the counters in front of its tile itself.  Forced here (wait of 0 cycles): the build must be the same,
    bit for bit against the oracle tree, and the default is restored afterwards."""
    from paper_1901_08088_b200 import qbvh
    from test_gpu_parity import check_build
    w = W.make_config(5)
    default = qbvh.qbvh_get_option(qbvh.OPT_DEBUG_SCAN_SPIN)
    assert default > 0
    try:
        qbvh.qbvh_set_option(qbvh.OPT_DEBUG_SCAN_SPIN, 0)
        out, t = check_build(w, 32)
        assert int(out["counts"][3]) == 6
    finally:
        qbvh.qbvh_set_option(qbvh.OPT_DEBUG_SCAN_SPIN, default)


def test_f64_and_range_enqueue_forms():
    """qbvh_neighbors_f64_enqueue / qbvh_neighbors_range_enqueue + qbvh_neighbors_result give what the synchronous calls
    give: M, counts, and the same rows as sets."""
    import torch
    from paper_1901_08088_b200 import qbvh
    w = W.make_config(3, small=True)
    nl = _built(w)
    first, count, cap = 777, 5000, w.max_neigh
    lst = [torch.full((count, cap), -1, dtype=torch.int32, device=nl.device) for _ in range(2)]
    cnt = [torch.full((count,), -1, dtype=torch.int32, device=nl.device) for _ in range(2)]
    M0 = qbvh.qbvh_neighbors_range(w.r_list, lst[0], cnt[0], cap, first, count)
    qbvh.qbvh_neighbors_range_enqueue(w.r_list, lst[1], cnt[1], cap, first, count)
    assert qbvh.qbvh_neighbors_result() == M0 and torch.equal(cnt[0], cnt[1])
    a, b, c = lst[0].cpu().numpy(), lst[1].cpu().numpy(), cnt[0].cpu().numpy()
    assert all(np.array_equal(np.sort(a[k, :c[k]]), np.sort(b[k, :c[k]])) for k in range(count))
    pos64, box64, r64 = W.as_f64(w)
    nl64 = qbvh.NeighborList(w.N, T=w.T, max_neigh=cap, device=nl.device)
    nl64.build(torch.from_numpy(pos64).to(nl.device), torch.from_numpy(w.type).to(nl.device), box64)
    M1 = nl64.neighbors(r64, retry=False)
    ref = nl64.n_neigh.clone()
    nl64.n_neigh.fill_(-1)
    nl64.neighbors_enqueue(r64)                                    # the fp64 form: the object was built from fp64 positions
    assert nl64.neighbors_result() == M1 and torch.equal(nl64.n_neigh, ref)
    rp, nb = ON.neighbor_list_f64(pos64, w.type, box64, r64)
    assert np.array_equal(ref.cpu().numpy()[: w.N], np.diff(rp))


@pytest.mark.parametrize("opt,value", [("OPT_GROUP_MAX", 16), ("OPT_GROUP_MAX", 5), ("OPT_CELL_LEVEL", 2), ("OPT_CELL_LEVEL", 6)])
def test_group_size_and_cell_level_do_not_change_tree_or_lists(opt, value):
    """QBVH_OPT_GROUP_MAX and QBVH_OPT_CELL_LEVEL are tuning knobs: whatever they are set to, the build products are the
    oracle tree bit for bit and the lists the oracle's."""
    from paper_1901_08088_b200 import qbvh
    from test_gpu_parity import check_build
    key = getattr(qbvh, opt)
    default = qbvh.qbvh_get_option(key)
    try:
        qbvh.qbvh_set_option(key, value)
        for cid in (2, 3):
            w = W.make_config(cid, small=True)
            out, t = check_build(w, 32)
            if opt == "OPT_CELL_LEVEL":
                lvl = value
                while (w.T << (3 * lvl)) > (1 << 18):            # the documented cap: T * 8^level <= 2^18
                    lvl -= 1
                assert int(out["counts"][3]) == lvl
            compare_with_oracle(w, out, ON.neighbor_list(w.pos, w.type, w.box, w.r_list))
    finally:
        qbvh.qbvh_set_option(key, default)
    with pytest.raises(qbvh.QbvhError):
        qbvh.qbvh_set_option(key, 33 if opt == "OPT_GROUP_MAX" else 7)


@pytest.mark.parametrize("world", [2, 3, 5])
@pytest.mark.parametrize("cid", [3, 5])
def test_slab_decomposition_emulated_on_one_gpu(cid, world):
    """SlabNeighborList with the CUDA backend, the ranks played one after another on one GPU (the exchange itself is
    covered over gloo in test_slab_host.py): own + halo particles in the original periodic box, rows of the own particles,
    entries mapped to global ids — merged over the ranks it must be the oracle's list of the whole system, exactly."""
    import torch
    from paper_1901_08088_b200 import qbvh, sharded
    w = W.make_config(cid, small=True)
    dev = torch.device("cuda:0")
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, 32)
    qbvh.qbvh_set_option(qbvh.OPT_STATS, 0)
    qbvh.qbvh_set_collapse_hint(None)
    snl = sharded.SlabNeighborList(w.box, w.r_list, T=w.T, max_neigh=16, device=dev)      # capacity too small: the retry path
    parts, ghosts_total = [], 0
    for g in range(world):
        own, ghosts = sharded.local_set_indices(w.pos, w.box, world, g, snl.h)
        idx = np.concatenate([own, ghosts])
        snl.build_from_local_set(torch.from_numpy(w.pos[idx]).to(dev), None if w.type is None else torch.from_numpy(w.type[idx]).to(dev),
                                 torch.from_numpy(idx.astype(np.int64)).to(dev), len(own), w.N)
        gid, n_neigh, nlist, M = snl.neighbors()
        parts.append((gid.cpu().numpy(), n_neigh.cpu().numpy(), nlist.cpu().numpy()))
        ghosts_total += len(ghosts)
    qbvh.qbvh_set_workspace(None)
    n_all, l_all = sharded.merge_slices(w.N, parts)
    out = {"M": int(n_all.max()), "max_neigh": l_all.shape[1], "nlist": l_all, "n_neigh": n_all}
    compare_with_oracle(w, out, ON.neighbor_list(w.pos, w.type, w.box, w.r_list))
    assert 0 < ghosts_total < 2 * w.N
