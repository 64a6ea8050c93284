"""qbvh_morton_keys_noalloc — the one entry point for callers that cannot allocate device memory.

Who needs it: code that lives inside another GPU program and only ever sees that program's buffers (a plugin called
from an MD engine's step loop), code under a framework whose memory pool already holds all of the HBM so that a plain
cudaMalloc fails, and loops where cudaMalloc/cudaFree are banned because they synchronise the device.  They cannot
hand the library a workspace, so this call keeps its working memory in an array compiled into libqbvh.so (393,472 bytes
per GPU, fixed, hence N <= 2^22) and every call re-uses it.

What is checked: its keys and frames are bitwise those of the ordinary workspace path (qbvh_build + debug export) on
the same input — integer and bit-pattern work, so the tolerance is zero, as in test_gpu_parity.py — on calls made back
to back, where each call finds the array as the previous one left it (a larger problem, then a smaller one in another
box with another number of types, then the first again).

This file sorts last on purpose (pytest -x stops at the first failure: a failure here must not hide the parity tests).
It passes alone in a fresh process and after the rest of the suite: it uses nothing of the library's global context
beyond what gpu_run sets up for the comparison path itself.
"""
import numpy as np
import pytest

from paper_1901_08088_b200 import workloads as W


def _existing_path(w):
    """Keys in input order and the frames, from the workspace path: qbvh_build, then the debug exports."""
    from gpu_util import gpu_run
    out = gpu_run(w, K=32, export=True)
    keys = np.empty(w.N, np.uint32)
    keys[out["perm"].astype(np.int64)] = out["keys_sorted"]       # key of sorted position k belongs to particle perm[k]
    return keys, out["frames"]


def _no_alloc(w, bufs):
    """One call of the new entry point into buffers that already exist (the caller 'cannot allocate')."""
    import torch
    from paper_1901_08088_b200 import qbvh
    pos, typ, keys, frames, status = bufs
    pos[: w.N].copy_(torch.from_numpy(w.pos))
    if w.type is not None:
        typ[: w.N].copy_(torch.from_numpy(w.type))
    keys.fill_(0x7FFFFFFF)
    frames.fill_(float("nan"))
    status.fill_(-1)
    rc = qbvh.qbvh_morton_keys_noalloc(pos, typ if w.type is not None else None, w.N, w.box, w.T, keys, frames, status,
                                       torch.cuda.current_stream().cuda_stream)
    assert rc == qbvh.OK
    torch.cuda.synchronize()
    return keys[: w.N].cpu().numpy().view(np.uint32), frames.cpu().numpy(), int(status.item())


def _compare(w, got, ref):
    keys, frames, status = got
    rkeys, rframes = ref
    assert status == 0
    assert np.array_equal(keys, rkeys)                                       # bit-exact, every particle
    counts = np.bincount(w.type, minlength=4) if w.type is not None else np.array([w.N, 0, 0, 0])
    for t in range(4):
        if counts[t] > 0:
            assert np.array_equal(frames[t, :9].view(np.uint32), rframes[t, :9].view(np.uint32)), t   # lo, hi, delta: bit patterns
            assert np.all(frames[t, 9:] == 0)
        else:
            assert np.all(frames[t] == 0)


@pytest.mark.gpu
def test_no_alloc_keys_and_frames_equal_the_workspace_path_on_calls_in_a_row():
    import torch
    dev = torch.device("cuda:0")
    a = W.lj_uniform(N=70001, rho=0.85, r_list=1.2, config_id=77)       # 69 blocks, ragged last one, T = 1
    b = W.make_config(3, small=True)                                   # two types, another box, fewer blocks
    c = W.shifted(W.lj_uniform(N=3001, rho=0.6, r_list=1.2, config_id=78), (3.5, -1.25, 10.0))   # box not centred
    refs = {id(w): _existing_path(w) for w in (a, b, c)}
    nmax = max(w.N for w in (a, b, c))
    # the caller's own buffers, made once up front; nothing is allocated around the calls below
    bufs = (torch.empty((nmax, 3), dtype=torch.float32, device=dev), torch.zeros(nmax, dtype=torch.int32, device=dev),
            torch.empty(nmax, dtype=torch.int32, device=dev), torch.empty((4, 12), dtype=torch.float32, device=dev),
            torch.empty(1, dtype=torch.int32, device=dev))
    for w in (a, b, a, c, c):                                          # each call inherits the previous call's scratch
        views = (bufs[0][: w.N], bufs[1][: w.N], bufs[2], bufs[3], bufs[4])
        _compare(w, _no_alloc(w, views), refs[id(w)])


@pytest.mark.gpu
def test_no_alloc_edge_cases():
    import torch
    from paper_1901_08088_b200 import qbvh
    dev = torch.device("cuda:0")
    box = np.array([-4, -4, -4, 8, 8, 8], np.float32)
    keys = torch.full((8,), 5, dtype=torch.int32, device=dev)
    frames = torch.full((4, 12), 7.0, dtype=torch.float32, device=dev)
    status = torch.full((1,), -1, dtype=torch.int32, device=dev)
    st = torch.cuda.current_stream().cuda_stream
    # N = 0: nothing to key, frames all zero
    assert qbvh.qbvh_morton_keys_noalloc(None, None, 0, box, 1, None, frames, status, st) == qbvh.OK
    torch.cuda.synchronize()
    assert status.item() == 0 and torch.all(frames == 0) and torch.all(keys == 5)
    # a type id outside [0, T): keyed as type 0 and reported in the status word; the next call starts clean again
    pos = torch.tensor([[0.5, 0.5, 0.5], [-3.0, 2.0, 1.0], [3.9, -4.0, 0.0]], dtype=torch.float32, device=dev)
    typ = torch.tensor([0, 5, 1], dtype=torch.int32, device=dev)
    assert qbvh.qbvh_morton_keys_noalloc(pos, typ, 3, box, 2, keys, frames, status, st) == qbvh.OK
    torch.cuda.synchronize()
    k = keys[:3].cpu().numpy().view(np.uint32)
    assert status.item() == 1 and (k >> 30).tolist() == [0, 0, 1] and torch.all(keys[3:] == 5)
    fr = frames.cpu().numpy()
    assert fr[0, :6].tolist() == [-3.0, 0.5, 0.5, 0.5, 2.0, 1.0] and fr[1, :6].tolist() == [3.9000000953674316, -4.0, 0.0] * 2
    assert np.all(fr[1, 6:9] == 0) and np.all(fr[2:] == 0)
    typ[1] = 1
    assert qbvh.qbvh_morton_keys_noalloc(pos, typ, 3, box, 2, keys, frames, status, st) == qbvh.OK
    torch.cuda.synchronize()
    assert status.item() == 0


def test_no_alloc_rejects_sizes_beyond_its_scratch():
    """Host-side checks come before any CUDA call, so this needs no device: N above the compiled-in limit is refused
    with its own error code and text, bad arguments as everywhere else."""
    from paper_1901_08088_b200 import qbvh
    box = np.array([0, 0, 0, 1, 1, 1], np.float32)
    fake = 4096                                                        # never dereferenced: the call returns first
    with pytest.raises(qbvh.QbvhError) as e:
        qbvh.qbvh_morton_keys_noalloc(fake, None, qbvh.NOALLOC_MAX_N + 1, box, 1, fake, fake, fake, None)
    assert e.value.code == qbvh.ERR_NOALLOC_LIMIT and "QBVH_NOALLOC_MAX_N" in str(e.value)
    for args in [(fake, None, -1, box, 1, fake, fake, fake), (fake, None, 10, box, 0, fake, fake, fake),
                 (fake, None, 10, box, 5, fake, fake, fake), (None, None, 10, box, 1, fake, fake, fake),
                 (fake, None, 10, box, 1, None, fake, fake), (fake, None, 10, box, 1, fake, None, fake),
                 (fake, None, 10, box, 1, fake, fake, None),
                 (fake, None, 10, np.array([0, 0, 0, 1, 0, 1], np.float32), 1, fake, fake, fake)]:
        with pytest.raises(qbvh.QbvhError) as e:
            qbvh.qbvh_morton_keys_noalloc(*args, None)
        assert e.value.code == qbvh.ERR_INVALID_ARG
