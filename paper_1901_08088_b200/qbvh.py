"""ctypes binding of libqbvh.so — same names as include/qbvh.h, argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C-ABI.  PyTorch is used for device memory
and streams.  Importing this module fails loudly if the CUDA library has not been built; there is no
CPU fallback.  Nothing here imports ``oracle/``.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqbvh.so")

OK = 0
ERR_INVALID_ARG, ERR_NOT_BUILT, ERR_WORKSPACE, ERR_CUTOFF_TOO_LARGE, ERR_TYPE_RANGE, ERR_CUDA, ERR_INTERNAL = -1, -2, -3, -4, -5, -6, -7
ERR_NOALLOC_LIMIT = -8
NOALLOC_MAX_N = 1 << 22
MAX_TYPES = 4
OPT_LEAF_COLLAPSE, OPT_STATS, OPT_VARIANT, OPT_DEBUG_BUILD_TAG, OPT_DEBUG_SCAN_SPIN, OPT_GROUP_MAX, OPT_CELL_LEVEL = 1, 2, 3, 4, 5, 6, 7
EXPORT_KEYS_SORTED, EXPORT_PERM, EXPORT_NODES, EXPORT_PARENT, EXPORT_FRAMES, EXPORT_SEGMENTS, EXPORT_SORTED_POS, EXPORT_COUNTS = range(1, 9)

# every symbol include/qbvh.h declares
SYMBOLS = ("qbvh_set_stream", "qbvh_set_num_types", "qbvh_workspace_bytes", "qbvh_set_workspace",
           "qbvh_set_option", "qbvh_get_option", "qbvh_build", "qbvh_neighbors", "qbvh_count_overlaps", "qbvh_staging_bytes",
           "qbvh_set_staging", "qbvh_build_host", "qbvh_neighbors_host", "qbvh_get_stats", "qbvh_debug_export",
           "qbvh_error_string", "qbvh_padded_radius", "qbvh_set_collapse_hint", "qbvh_build_f64", "qbvh_neighbors_f64", "qbvh_last_d2h_bytes", "qbvh_neighbors_range",
           "qbvh_neighbors_enqueue", "qbvh_neighbors_result", "qbvh_morton_keys_noalloc", "qbvh_padded_radius_sq",
           "qbvh_neighbors_f64_enqueue", "qbvh_neighbors_range_enqueue")


class QbvhStats(C.Structure):
    _fields_ = [("node_tests", C.c_uint64), ("leaf_overlaps", C.c_uint64), ("dist_checks", C.c_uint64),
                ("neighbors", C.c_uint64), ("images", C.c_uint64),
                ("groups", C.c_uint64), ("group_node_tests", C.c_uint64), ("group_leaf_hits", C.c_uint64),
                ("group_candidates", C.c_uint64), ("group_dist_checks", C.c_uint64), ("group_walk_steps", C.c_uint64)]


class QbvhError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {qbvh_error_string(code)} ({code})")


if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1901_08088_b200.build` "
                      "(there is no CPU fallback)")
_lib = C.CDLL(LIB_PATH)
_vp, _i32, _i64 = C.c_void_p, C.c_int32, C.c_int64
_lib.qbvh_set_stream.argtypes = [_vp]
_lib.qbvh_set_num_types.argtypes = [_i32]
_lib.qbvh_workspace_bytes.argtypes = [_i64, _i32]
_lib.qbvh_workspace_bytes.restype = _i64
_lib.qbvh_set_workspace.argtypes = [_vp, _i64]
_lib.qbvh_set_option.argtypes = [_i32, _i32]
_lib.qbvh_get_option.argtypes = [_i32]
_lib.qbvh_set_collapse_hint.argtypes = [_vp, _i32]
_lib.qbvh_build.argtypes = [_vp, _vp, _i64, _vp]
_lib.qbvh_neighbors.argtypes = [_vp, _vp, _vp, _i32]
_lib.qbvh_neighbors_enqueue.argtypes = [_vp, _vp, _vp, _i32]
_lib.qbvh_neighbors_result.argtypes = []
_lib.qbvh_neighbors_f64_enqueue.argtypes = [_vp, _vp, _vp, _i32]
_lib.qbvh_neighbors_range_enqueue.argtypes = [_vp, _vp, _vp, _i32, _i64, _i64]
_lib.qbvh_count_overlaps.argtypes = [_vp, _vp]
_lib.qbvh_neighbors_range.argtypes = [_vp, _vp, _vp, _i32, _i64, _i64]
_lib.qbvh_build_f64.argtypes = [_vp, _vp, _i64, _vp]
_lib.qbvh_neighbors_f64.argtypes = [_vp, _vp, _vp, _i32]
_lib.qbvh_staging_bytes.argtypes = [_i64, _i32]
_lib.qbvh_staging_bytes.restype = _i64
_lib.qbvh_set_staging.argtypes = [_vp, _i64]
_lib.qbvh_build_host.argtypes = [_vp, _vp, _i64, _vp]
_lib.qbvh_neighbors_host.argtypes = [_vp, _vp, _vp, _i32]
_lib.qbvh_last_d2h_bytes.argtypes = []
_lib.qbvh_last_d2h_bytes.restype = _i64
_lib.qbvh_get_stats.argtypes = [C.POINTER(QbvhStats)]
_lib.qbvh_debug_export.argtypes = [_i32, _vp, _i64]
_lib.qbvh_debug_export.restype = _i64
_lib.qbvh_padded_radius.argtypes = [C.c_float, _vp]
_lib.qbvh_padded_radius.restype = C.c_float
_lib.qbvh_morton_keys_noalloc.argtypes = [_vp, _vp, _i64, _vp, _i32, _vp, _vp, _vp, _vp]
_lib.qbvh_padded_radius_sq.argtypes = [C.c_float, _vp]
_lib.qbvh_padded_radius_sq.restype = C.c_float
_lib.qbvh_error_string.argtypes = [C.c_int]
_lib.qbvh_error_string.restype = C.c_char_p


def _ptr(x):
    """Device/host pointer of a torch tensor, numpy array, int or None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        assert x.flags["C_CONTIGUOUS"]
        return x.ctypes.data
    assert x.is_contiguous()
    return x.data_ptr()


_bound_workspace = None   # (id of the NeighborList, device pointer) the C context currently points at
_num_types = 1   # T of the last qbvh_set_num_types: the C side reads T x T floats from r_list_ij


def _r_list(r_list_ij):
    """HOST T x T fp32 cutoff table; the size is checked here because the C-ABI takes a bare pointer."""
    r = np.ascontiguousarray(r_list_ij, dtype=np.float32)
    if r.size != _num_types * _num_types:
        raise ValueError(f"r_list_ij holds {r.size} values; qbvh_set_num_types({_num_types}) needs {_num_types}x{_num_types}")
    return r


def _host_f32(a, n):
    a = np.ascontiguousarray(a, dtype=np.float32).reshape(-1)
    assert a.size == n, (a.size, n)
    return a


def qbvh_error_string(code: int) -> str:
    return _lib.qbvh_error_string(int(code)).decode()


def _check(rc: int, where: str) -> int:
    if rc < 0:
        raise QbvhError(int(rc), where)
    return int(rc)


def qbvh_set_stream(cuda_stream: int) -> int:
    return _check(_lib.qbvh_set_stream(cuda_stream), "qbvh_set_stream")


def qbvh_set_num_types(T: int) -> int:
    global _num_types
    rc = _check(_lib.qbvh_set_num_types(T), "qbvh_set_num_types")
    _num_types = int(T)
    return rc


def qbvh_workspace_bytes(N: int, T: int = 1) -> int:
    return _check(_lib.qbvh_workspace_bytes(N, T), "qbvh_workspace_bytes")


def qbvh_set_workspace(buf, nbytes: int | None = None) -> int:
    global _bound_workspace
    _bound_workspace = None
    if nbytes is None:
        nbytes = 0 if buf is None else buf.numel() * buf.element_size()
    return _check(_lib.qbvh_set_workspace(_ptr(buf), nbytes), "qbvh_set_workspace")


def qbvh_set_option(key: int, value: int) -> int:
    return _check(_lib.qbvh_set_option(key, value), "qbvh_set_option")


def qbvh_set_collapse_hint(r_hint) -> int:
    """r_hint: per-type expected query radius (HOST, at most MAX_TYPES values) or None for no hint."""
    if r_hint is None:
        return _check(_lib.qbvh_set_collapse_hint(None, 0), "qbvh_set_collapse_hint")
    r = np.ascontiguousarray(r_hint, dtype=np.float32).reshape(-1)
    return _check(_lib.qbvh_set_collapse_hint(r.ctypes.data, r.size), "qbvh_set_collapse_hint")


def qbvh_get_option(key: int) -> int:
    return _check(_lib.qbvh_get_option(key), "qbvh_get_option")


def qbvh_build(pos, type, N: int, box) -> int:
    """pos, type: DEVICE tensors (float32 N x 3, int32 N or None); box: 6 host floats."""
    box = _host_f32(box, 6)
    return _check(_lib.qbvh_build(_ptr(pos), _ptr(type), N, box.ctypes.data), "qbvh_build")


def qbvh_neighbors(r_list_ij, nlist, n_neigh, max_neigh: int) -> int:
    """r_list_ij: host T x T; nlist, n_neigh: DEVICE int32 tensors.  Returns M = max n_neigh (overflow iff M > max_neigh)."""
    r = _r_list(r_list_ij)
    return _check(_lib.qbvh_neighbors(r.ctypes.data, _ptr(nlist), _ptr(n_neigh), max_neigh), "qbvh_neighbors")


def qbvh_neighbors_enqueue(r_list_ij, nlist, n_neigh, max_neigh: int) -> None:
    """qbvh_neighbors without the wait: the traversal is enqueued on the stream; take M with qbvh_neighbors_result."""
    r = _r_list(r_list_ij)
    _check(_lib.qbvh_neighbors_enqueue(r.ctypes.data, _ptr(nlist), _ptr(n_neigh), max_neigh), "qbvh_neighbors_enqueue")


def qbvh_neighbors_f64_enqueue(r_list_ij, nlist, n_neigh, max_neigh: int) -> None:
    """qbvh_neighbors_f64 without the wait; M comes from qbvh_neighbors_result."""
    r = np.ascontiguousarray(r_list_ij, dtype=np.float64)
    if r.size != _num_types * _num_types:
        raise ValueError(f"r_list_ij holds {r.size} values; qbvh_set_num_types({_num_types}) needs {_num_types}x{_num_types}")
    _check(_lib.qbvh_neighbors_f64_enqueue(r.ctypes.data, _ptr(nlist), _ptr(n_neigh), max_neigh), "qbvh_neighbors_f64_enqueue")


def qbvh_neighbors_range_enqueue(r_list_ij, nlist, n_neigh, max_neigh: int, first: int, count: int) -> None:
    """qbvh_neighbors_range without the wait; the maximum over the range comes from qbvh_neighbors_result."""
    r = _r_list(r_list_ij)
    _check(_lib.qbvh_neighbors_range_enqueue(r.ctypes.data, _ptr(nlist), _ptr(n_neigh), max_neigh, first, count),
           "qbvh_neighbors_range_enqueue")


def qbvh_neighbors_result() -> int:
    """Synchronises the stream; M of the last qbvh_neighbors_enqueue."""
    return _check(_lib.qbvh_neighbors_result(), "qbvh_neighbors_result")


def qbvh_neighbors_range(r_list_ij, nlist, n_neigh, max_neigh: int, first: int, count: int) -> int:
    """Lists of the particles at sorted positions [first, first + count) only (row k = sorted position first + k)."""
    r = _r_list(r_list_ij)
    return _check(_lib.qbvh_neighbors_range(r.ctypes.data, _ptr(nlist), _ptr(n_neigh), max_neigh, first, count),
                  "qbvh_neighbors_range")


def qbvh_build_f64(pos, type, N: int, box) -> int:
    """pos: DEVICE float64 N x 3; type: DEVICE int32 N or None; box: 6 host doubles."""
    box = np.ascontiguousarray(box, dtype=np.float64).reshape(-1)
    assert box.size == 6
    return _check(_lib.qbvh_build_f64(_ptr(pos), _ptr(type), N, box.ctypes.data), "qbvh_build_f64")


def qbvh_neighbors_f64(r_list_ij, nlist, n_neigh, max_neigh: int) -> int:
    """r_list_ij: host T x T float64; otherwise as qbvh_neighbors."""
    r = np.ascontiguousarray(r_list_ij, dtype=np.float64)
    if r.size != _num_types * _num_types:
        raise ValueError(f"r_list_ij holds {r.size} values; qbvh_set_num_types({_num_types}) needs {_num_types}x{_num_types}")
    return _check(_lib.qbvh_neighbors_f64(r.ctypes.data, _ptr(nlist), _ptr(n_neigh), max_neigh), "qbvh_neighbors_f64")


def qbvh_count_overlaps(r_list_ij, n_overlap) -> int:
    """The paper's accept-on-leaf-overlap count.  n_overlap: DEVICE int32 tensor of N."""
    r = _r_list(r_list_ij)
    return _check(_lib.qbvh_count_overlaps(r.ctypes.data, _ptr(n_overlap)), "qbvh_count_overlaps")


def qbvh_staging_bytes(N: int, max_neigh: int) -> int:
    return _check(_lib.qbvh_staging_bytes(N, max_neigh), "qbvh_staging_bytes")


def qbvh_set_staging(buf, nbytes: int | None = None) -> int:
    if nbytes is None:
        nbytes = 0 if buf is None else buf.numel() * buf.element_size()
    return _check(_lib.qbvh_set_staging(_ptr(buf), nbytes), "qbvh_set_staging")


def qbvh_build_host(pos, type, N: int, box) -> int:
    """pos, type: HOST buffers (numpy arrays or pinned CPU torch tensors)."""
    box = _host_f32(box, 6)
    return _check(_lib.qbvh_build_host(_ptr(pos), _ptr(type), N, box.ctypes.data), "qbvh_build_host")


def qbvh_neighbors_host(r_list_ij, nlist, n_neigh, max_neigh: int) -> int:
    r = _r_list(r_list_ij)
    return _check(_lib.qbvh_neighbors_host(r.ctypes.data, _ptr(nlist), _ptr(n_neigh), max_neigh), "qbvh_neighbors_host")


def qbvh_padded_radius(r: float, box) -> float:
    """Host arithmetic only (no device): the padded pruning radius of include/qbvh.h."""
    box = _host_f32(box, 6)
    v = float(_lib.qbvh_padded_radius(C.c_float(float(r)), box.ctypes.data))
    if v < 0:
        raise QbvhError(ERR_INVALID_ARG, "qbvh_padded_radius")
    return v


def qbvh_morton_keys_noalloc(pos, type, N: int, box, T: int, keys, frames, status, cuda_stream: int | None = None) -> int:
    """Morton keys + per-type root frames with no workspace and no allocation (include/qbvh.h): for callers that
    cannot obtain device memory themselves.  pos, type, keys (uint32/int32 N), frames (float32 4 x 12), status
    (int32 1): DEVICE tensors the caller already has; box: 6 host floats.  N <= NOALLOC_MAX_N.  Asynchronous."""
    box = _host_f32(box, 6)
    return _check(_lib.qbvh_morton_keys_noalloc(_ptr(pos), _ptr(type), N, box.ctypes.data, T, _ptr(keys), _ptr(frames),
                                                _ptr(status), cuda_stream), "qbvh_morton_keys_noalloc")


def qbvh_padded_radius_sq(r: float, box) -> float:
    """Host arithmetic only: the squared padded pruning radius, rounded up, as the kernels receive it."""
    box = _host_f32(box, 6)
    v = float(_lib.qbvh_padded_radius_sq(C.c_float(float(r)), box.ctypes.data))
    if v < 0:
        raise QbvhError(ERR_INVALID_ARG, "qbvh_padded_radius_sq")
    return v


def qbvh_last_d2h_bytes() -> int:
    return int(_lib.qbvh_last_d2h_bytes())


def qbvh_get_stats() -> dict:
    s = QbvhStats()
    _check(_lib.qbvh_get_stats(C.byref(s)), "qbvh_get_stats")
    return {k: int(getattr(s, k)) for k, _ in QbvhStats._fields_}


def qbvh_debug_export(what: int, N: int) -> np.ndarray:
    """Host copy of a build product (see QBVH_EXPORT_* in include/qbvh.h)."""
    shapes = {EXPORT_KEYS_SORTED: (np.uint32, (N,)), EXPORT_PERM: (np.uint32, (N,)),
              EXPORT_NODES: (np.int32, (max(2 * N - 1, 0), 4)), EXPORT_PARENT: (np.int32, (max(2 * N - 1, 0),)),
              EXPORT_FRAMES: (np.float32, (4, 12)), EXPORT_SEGMENTS: (np.int32, (10,)),
              EXPORT_SORTED_POS: (np.float32, (N, 4)), EXPORT_COUNTS: (np.int32, (4,))}
    dt, shp = shapes[what]
    out = np.zeros(shp, dt)
    avail = _check(_lib.qbvh_debug_export(what, out.ctypes.data, out.nbytes), "qbvh_debug_export")
    assert avail == out.nbytes, (avail, out.nbytes)
    return out


def qbvh_debug_export_into(what: int, dst) -> int:
    """Array build products (EXPORT_KEYS_SORTED, PERM, NODES, PARENT, FRAMES, SORTED_POS) copied into an existing tensor
    or array `dst`, on the host or on the device; returns the bytes available."""
    nbytes = dst.nbytes if isinstance(dst, np.ndarray) else dst.numel() * dst.element_size()
    return _check(_lib.qbvh_debug_export(what, _ptr(dst), nbytes), "qbvh_debug_export")


# ---------------------------------------------------------------------------------------------------------
# Convenience wrapper: owns the torch workspace, retries on overflow.  Plumbing only — no arithmetic.
# ---------------------------------------------------------------------------------------------------------
class NeighborList:
    """Device-resident Verlet list builder.

    >>> nl = NeighborList(N, T=1, max_neigh=128)
    >>> nl.build(pos_cuda, None, box)              # qbvh_build
    >>> M = nl.neighbors(r_list)                   # qbvh_neighbors (+ re-allocation and retry on overflow)
    >>> nl.nlist, nl.n_neigh                       # int32 CUDA tensors
    """

    def __init__(self, N: int, T: int = 1, max_neigh: int = 128, device="cuda:0"):
        import torch
        self.torch = torch
        self.device = torch.device(device)
        self.N, self.T, self.max_neigh = int(N), int(T), int(max_neigh)
        self.workspace = torch.empty(qbvh_workspace_bytes(N, T), dtype=torch.uint8, device=self.device)
        self.nlist = torch.empty((max(N, 1), max(max_neigh, 1)), dtype=torch.int32, device=self.device)
        self.n_neigh = torch.zeros(max(N, 1), dtype=torch.int32, device=self.device)
        self.retries = 0

    def _activate(self):
        """Point the process-global context at this object: stream, T and (only when it changed) the workspace —
        qbvh_set_workspace restarts the build tags, i.e. costs a clear of the meeting slots at the next build."""
        global _bound_workspace
        qbvh_set_stream(self.torch.cuda.current_stream(self.device).cuda_stream)
        qbvh_set_num_types(self.T)
        if _bound_workspace != (id(self), self.workspace.data_ptr()):
            qbvh_set_workspace(self.workspace)
            _bound_workspace = (id(self), self.workspace.data_ptr())

    def release(self):
        """Detach the library from this object's workspace (the tree is gone afterwards)."""
        global _bound_workspace
        if _bound_workspace is not None and _bound_workspace[0] == id(self):
            _bound_workspace = None
            qbvh_set_workspace(None)

    def __del__(self):
        try:
            self.release()
        except Exception:
            pass

    def build(self, pos, type, box):
        """pos: CUDA float32 (qbvh_build) or float64 (qbvh_build_f64) N x 3."""
        assert pos.is_cuda and pos.dtype in (self.torch.float32, self.torch.float64) and tuple(pos.shape) == (self.N, 3)
        assert type is None or (type.is_cuda and type.dtype == self.torch.int32)
        self._activate()
        self.f64 = pos.dtype == self.torch.float64
        return (qbvh_build_f64 if self.f64 else qbvh_build)(pos, type, self.N, box)

    def neighbors_enqueue(self, r_list) -> None:
        """Lists without the wait (qbvh_neighbors_enqueue / qbvh_neighbors_f64_enqueue); M comes from neighbors_result()."""
        call = qbvh_neighbors_f64_enqueue if getattr(self, "f64", False) else qbvh_neighbors_enqueue
        call(r_list, self.nlist, self.n_neigh, self.max_neigh)

    def neighbors_result(self) -> int:
        return qbvh_neighbors_result()

    def neighbors(self, r_list, retry: bool = True) -> int:
        call = qbvh_neighbors_f64 if getattr(self, "f64", False) else qbvh_neighbors
        M = call(r_list, self.nlist, self.n_neigh, self.max_neigh)
        while retry and M > self.max_neigh:
            self.retries += 1
            self.max_neigh = int((M + 7) // 8 * 8)
            self.nlist = self.torch.empty((max(self.N, 1), self.max_neigh), dtype=self.torch.int32, device=self.device)
            M = call(r_list, self.nlist, self.n_neigh, self.max_neigh)
        return M
