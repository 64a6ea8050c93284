"""ORACLE — TEST INFRASTRUCTURE ONLY.  ctypes glue around oracle/tree.c.

CPU restatements of build steps a1..a6 and of Algorithm 1 (a7, a8), see tree.c.
The sort (a2) is `numpy.argsort(kind="stable")` — a library routine serving as a
step (ascending key, ties by original index; "sorted along a Z-order curve").
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import build as _build

_lib = None
_f32p, _i32p, _i64p, _u32p = (C.POINTER(C.c_float), C.POINTER(C.c_int32), C.POINTER(C.c_int64),
                              C.POINTER(C.c_uint32))


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.oracle_morton_keys.restype = None
        L.oracle_morton_keys.argtypes = [_f32p, _i32p, C.c_int64, _f32p, _u32p]
        L.oracle_build_tree.restype = None
        L.oracle_build_tree.argtypes = [_u32p, C.c_int64, _i64p, C.c_int32] + [_i32p] * 7
        L.oracle_fit_quantize.restype = None
        L.oracle_fit_quantize.argtypes = [_f32p, C.c_int64, _i64p, C.c_int32, _i32p, _i32p, _i32p, _f32p, _f32p,
                                          _f32p, _u32p, _u32p, _f32p, C.c_int]
        L.oracle_decompress_tables.restype = None
        L.oracle_decompress_tables.argtypes = [C.c_float, C.c_float, _f32p, _f32p]
        L.oracle_frame_delta.restype = C.c_float
        L.oracle_frame_delta.argtypes = [C.c_float, C.c_float]
        L.oracle_qlo_scan.restype = C.c_int
        L.oracle_qlo_scan.argtypes = [_f32p, C.c_float]
        L.oracle_qhi_scan.restype = C.c_int
        L.oracle_qhi_scan.argtypes = [_f32p, C.c_float]
        L.oracle_pad_abs.restype = C.c_float
        L.oracle_pad_abs.argtypes = [_f32p]
        L.oracle_r_pad.restype = C.c_float
        L.oracle_r_pad.argtypes = [C.c_float, C.c_float]
        L.oracle_R2.restype = C.c_float
        L.oracle_R2.argtypes = [C.c_float, C.c_float]
        L.oracle_traverse_fp32_boxes.restype = C.c_int64
        L.oracle_traverse_fp32_boxes.argtypes = [_f32p, C.c_int64, _i64p, C.c_int32, _f32p, _f32p, _f32p, _f32p, _i32p, _i32p,
                                                 _i32p, _i32p, _i64p, _i32p]
        L.oracle_traverse.restype = C.c_int64
        L.oracle_traverse.argtypes = [_f32p, C.c_int64, _i64p, C.c_int32, _f32p, _f32p, _u32p, _u32p, _i32p, _i32p,
                                      _i32p, _f32p, _i32p, _i64p, _i32p, _i64p, _i32p]
        _lib = L
    return _lib


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def morton_keys(pos, type, box) -> np.ndarray:
    pos = np.ascontiguousarray(pos, np.float32)
    type = None if type is None else np.ascontiguousarray(type, np.int32)
    box = np.ascontiguousarray(box, np.float32)
    key = np.zeros(max(len(pos), 1), np.uint32)
    lib().oracle_morton_keys(_p(pos, C.c_float), _p(type, C.c_int32), len(pos), _p(box, C.c_float),
                             _p(key, C.c_uint32))
    return key[:len(pos)]


def decompress_tables(lo: float, delta: float):
    Dlo = np.zeros(1024, np.float32)
    Dhi = np.zeros(1024, np.float32)
    lib().oracle_decompress_tables(C.c_float(lo), C.c_float(delta), _p(Dlo, C.c_float), _p(Dhi, C.c_float))
    return Dlo, Dhi


def frame_delta(lo: float, hi: float) -> np.float32:
    return np.float32(lib().oracle_frame_delta(C.c_float(lo), C.c_float(hi)))


def qlo_scan(Dlo, a) -> int:
    return int(lib().oracle_qlo_scan(_p(np.ascontiguousarray(Dlo, np.float32), C.c_float), C.c_float(a)))


def qhi_scan(Dhi, b) -> int:
    return int(lib().oracle_qhi_scan(_p(np.ascontiguousarray(Dhi, np.float32), C.c_float), C.c_float(b)))


def r_pad(r: float, box) -> np.float32:
    box = np.ascontiguousarray(box, np.float32)
    pad_abs = lib().oracle_pad_abs(_p(box, C.c_float))
    return np.float32(lib().oracle_r_pad(C.c_float(r), C.c_float(pad_abs)))


def R2_pad(r: float, box) -> np.float32:
    """Squared padded pruning radius, rounded up: the right-hand side of the sphere/box tests of the replay."""
    box = np.ascontiguousarray(box, np.float32)
    pad_abs = lib().oracle_pad_abs(_p(box, C.c_float))
    return np.float32(lib().oracle_R2(C.c_float(r), C.c_float(pad_abs)))


@dataclass
class RefTree:
    N: int
    T: int
    key: np.ndarray          # (N,) uint32, unsorted
    key_sorted: np.ndarray   # (N,) uint32
    perm: np.ndarray         # (N,) int64: sorted position k holds original particle perm[k]
    seg: np.ndarray          # (T+1,) int64
    pos_sorted: np.ndarray   # (N,3) float32
    left: np.ndarray
    right: np.ndarray
    rope: np.ndarray
    parent: np.ndarray
    first: np.ndarray
    last: np.ndarray
    roots: np.ndarray        # (T,) int32
    frames: np.ndarray       # (T,9) float32 {lo, hi, delta}
    blo: np.ndarray          # (2N-1,3) fp32 boxes
    bhi: np.ndarray
    wlo: np.ndarray          # (2N-1,) uint32 packed quantized lower bounds
    whi: np.ndarray
    tables: np.ndarray       # (T,2,3,1024) float32 decompression tables

    def nodes_int4(self) -> np.ndarray:
        """(2N-1,4) int32 {lo, hi, left, rope} — the 16-byte node of PAPER.md Fig. 3b."""
        out = np.empty((2 * self.N - 1, 4), np.int32)
        out[:, 0] = self.wlo.view(np.int32)
        out[:, 1] = self.whi.view(np.int32)
        out[:, 2] = self.left
        out[:, 3] = self.rope
        return out


def build(pos, type, box, T: int = 1, use_scan: bool = False) -> RefTree:
    pos = np.ascontiguousarray(pos, np.float32)
    N = len(pos)
    assert N >= 1
    box = np.ascontiguousarray(box, np.float32)
    key = morton_keys(pos, type, box)                     # a1
    perm = np.argsort(key, kind="stable")                 # a2
    key_sorted = np.ascontiguousarray(key[perm])
    seg = np.searchsorted(key_sorted >> np.uint32(30), np.arange(T + 1), side="left").astype(np.int64)
    pos_sorted = np.ascontiguousarray(pos[perm])          # a2'
    M = 2 * N - 1
    i32 = lambda: np.zeros(M, np.int32)
    left, right, rope, parent, first, last = i32(), i32(), i32(), i32(), i32(), i32()
    roots = np.zeros(T, np.int32)
    L = lib()
    L.oracle_build_tree(_p(key_sorted, C.c_uint32), N, _p(seg, C.c_int64), T, _p(left, C.c_int32),
                        _p(right, C.c_int32), _p(rope, C.c_int32), _p(parent, C.c_int32), _p(first, C.c_int32),
                        _p(last, C.c_int32), _p(roots, C.c_int32))          # a3 + a4
    frames = np.zeros((T, 9), np.float32)
    blo = np.zeros((M, 3), np.float32)
    bhi = np.zeros((M, 3), np.float32)
    wlo = np.zeros(M, np.uint32)
    whi = np.zeros(M, np.uint32)
    tables = np.zeros((T, 2, 3, 1024), np.float32)
    L.oracle_fit_quantize(_p(pos_sorted, C.c_float), N, _p(seg, C.c_int64), T, _p(left, C.c_int32),
                          _p(right, C.c_int32), _p(roots, C.c_int32), _p(frames, C.c_float), _p(blo, C.c_float),
                          _p(bhi, C.c_float), _p(wlo, C.c_uint32), _p(whi, C.c_uint32), _p(tables, C.c_float),
                          int(use_scan))                                      # a5 + a6
    return RefTree(N, T, key, key_sorted, perm, seg, pos_sorted, left, right, rope, parent, first, last, roots,
                   frames, blo, bhi, wlo, whi, tables)


def traverse(tree: RefTree, box, r_list, fill: bool = False):
    """Algorithm 1 in the paper's accept-on-leaf-overlap mode.  Returns a dict with per-sorted-particle
    n_overlap, n_tests, n_images and (fill=True) CSR candidate lists of sorted positions."""
    box = np.ascontiguousarray(box, np.float32)
    r_list = np.ascontiguousarray(r_list, np.float32)
    N, T = tree.N, tree.T
    n_overlap = np.zeros(N, np.int32)
    n_tests = np.zeros(N, np.int64)
    n_images = np.zeros(N, np.int32)
    args = [_p(tree.pos_sorted, C.c_float), N, _p(tree.seg, C.c_int64), T, _p(box, C.c_float),
            _p(r_list, C.c_float), _p(tree.wlo, C.c_uint32), _p(tree.whi, C.c_uint32), _p(tree.left, C.c_int32),
            _p(tree.rope, C.c_int32), _p(tree.roots, C.c_int32), _p(tree.tables, C.c_float)]
    total = lib().oracle_traverse(*args, _p(n_overlap, C.c_int32), _p(n_tests, C.c_int64), _p(n_images, C.c_int32),
                                  None, None)
    out = {"n_overlap": n_overlap, "n_tests": n_tests, "n_images": n_images, "total": int(total)}
    if fill:
        row_ptr = np.zeros(N + 1, np.int64)
        np.cumsum(n_overlap, out=row_ptr[1:])
        cand = np.zeros(max(int(total), 1), np.int32)
        lib().oracle_traverse(*args, _p(n_overlap, C.c_int32), _p(n_tests, C.c_int64), _p(n_images, C.c_int32),
                              _p(row_ptr, C.c_int64), _p(cand, C.c_int32))
        out["row_ptr"] = row_ptr
        out["cand"] = cand[:total]
    return out


def traverse_fp32_boxes(tree: RefTree, box, r_list):
    """Algorithm 1 on the tree's unquantized fp32 boxes (count pass): the census the quantized one is compared with
    to count the extra false-positive AABB tests of quantization."""
    box = np.ascontiguousarray(box, np.float32)
    r_list = np.ascontiguousarray(r_list, np.float32)
    N, T = tree.N, tree.T
    n_overlap = np.zeros(N, np.int32)
    n_tests = np.zeros(N, np.int64)
    n_images = np.zeros(N, np.int32)
    blo, bhi = np.ascontiguousarray(tree.blo, np.float32), np.ascontiguousarray(tree.bhi, np.float32)
    total = lib().oracle_traverse_fp32_boxes(_p(tree.pos_sorted, C.c_float), N, _p(tree.seg, C.c_int64), T, _p(box, C.c_float),
                                             _p(r_list, C.c_float), _p(blo, C.c_float), _p(bhi, C.c_float),
                                             _p(tree.left, C.c_int32), _p(tree.rope, C.c_int32), _p(tree.roots, C.c_int32),
                                             _p(n_overlap, C.c_int32), _p(n_tests, C.c_int64), _p(n_images, C.c_int32))
    return {"n_overlap": n_overlap, "n_tests": n_tests, "n_images": n_images, "total": int(total)}
