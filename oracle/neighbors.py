"""ORACLE — TEST INFRASTRUCTURE ONLY.  ctypes glue around oracle/neighbors.c.

`neighbor_list` returns the Verlet list of PAPER.md:31 under the periodic
boundaries of PAPER.md:166 as CSR arrays (row_ptr, nbr, band): row i holds the
ascending original indices j != i with O1(i,j) true; band[k] = 1 for pairs whose
exact (fp64) minimum-image distance lies within 1e-5 sigma of the cutoff.
"""
from __future__ import annotations

import ctypes as C
import os
import time

import numpy as np

from . import build as _build

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        f32p, i32p, i64p, u8p = (C.POINTER(C.c_float), C.POINTER(C.c_int32), C.POINTER(C.c_int64),
                                 C.POINTER(C.c_uint8))
        for name in ("oracle_brute_force", "oracle_cell_list"):
            fn = getattr(_lib, name)
            fn.restype = C.c_int64
            fn.argtypes = [f32p, i32p, C.c_int64, f32p, f32p, C.c_int32, i32p, i64p, i32p, u8p]
        _lib.oracle_pair.restype = C.c_int
        _lib.oracle_pair.argtypes = [f32p, f32p, f32p, C.c_float, f32p, C.POINTER(C.c_double)]
        _lib.oracle_num_threads.restype = C.c_int
        f64p = C.POINTER(C.c_double)
        for name in ("oracle_brute_force_f64", "oracle_cell_list_f64"):
            fn = getattr(_lib, name)
            fn.restype = C.c_int64
            fn.argtypes = [f64p, i32p, C.c_int64, f64p, f64p, C.c_int32, i32p, i64p, i32p]
        _lib.oracle_pair_f64.restype = C.c_int
        _lib.oracle_pair_f64.argtypes = [f64p, f64p, f64p, C.c_double, f64p]
    return _lib


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def num_threads() -> int:
    """Threads the OpenMP loops will use, capped by the CPUs this process may run on."""
    n = lib().oracle_num_threads()
    try:
        n = min(n, len(os.sched_getaffinity(0)))
    except AttributeError:
        pass
    return int(n)


def pair(pi, pj, box, r):
    """O1 on one pair: returns (is_neighbor, d2_fp32, d_fp64)."""
    pi = np.ascontiguousarray(pi, np.float32)
    pj = np.ascontiguousarray(pj, np.float32)
    box = np.ascontiguousarray(box, np.float32)
    d2 = C.c_float()
    d64 = C.c_double()
    ok = lib().oracle_pair(_p(pi, C.c_float), _p(pj, C.c_float), _p(box, C.c_float), C.c_float(float(r)),
                           C.byref(d2), C.byref(d64))
    return bool(ok), float(d2.value), float(d64.value)


def neighbor_list(pos, type, box, r_list, method: str = "auto", with_band: bool = True, timing: dict | None = None):
    """CSR neighbor list by the definition.  method: 'brute' | 'cell' | 'auto' (brute for N <= 16384)."""
    pos = np.ascontiguousarray(pos, np.float32)
    N = pos.shape[0]
    assert pos.shape == (N, 3)
    type = None if type is None else np.ascontiguousarray(type, np.int32)
    box = np.ascontiguousarray(box, np.float32)
    r_list = np.ascontiguousarray(r_list, np.float32)
    T = r_list.shape[0]
    assert r_list.shape == (T, T)
    if type is not None and N:
        assert type.min() >= 0 and type.max() < T
    if method == "auto":
        method = "brute" if N <= 16384 else "cell"
    fn = {"brute": lib().oracle_brute_force, "cell": lib().oracle_cell_list}[method]
    t0 = time.perf_counter()
    n_neigh = np.zeros(max(N, 1), np.int32)
    total = fn(_p(pos, C.c_float), _p(type, C.c_int32), N, _p(box, C.c_float), _p(r_list, C.c_float), T,
               _p(n_neigh, C.c_int32), None, None, None)
    assert total >= 0
    n_neigh = n_neigh[:N]
    row_ptr = np.zeros(N + 1, np.int64)
    np.cumsum(n_neigh, out=row_ptr[1:])
    nbr = np.empty(max(int(total), 1), np.int32)
    band = np.zeros(max(int(total), 1), np.uint8) if with_band else None
    total2 = fn(_p(pos, C.c_float), _p(type, C.c_int32), N, _p(box, C.c_float), _p(r_list, C.c_float), T,
                _p(n_neigh if N else np.zeros(1, np.int32), C.c_int32), _p(row_ptr, C.c_int64),
                _p(nbr, C.c_int32), _p(band, C.c_uint8))
    assert total2 == total
    if timing is not None:
        timing["seconds"] = time.perf_counter() - t0
        timing["threads"] = num_threads()
        timing["method"] = method
    return row_ptr, nbr[:total], (band[:total] if with_band else None)


def counts(pos, type, box, r_list, method: str = "auto") -> np.ndarray:
    row_ptr, _, _ = neighbor_list(pos, type, box, r_list, method=method, with_band=False)
    return np.diff(row_ptr).astype(np.int32)


# ---------------------------------------------------------------------------------------------------------
# double-precision particle data (oracle/neighbors_f64.c)
# ---------------------------------------------------------------------------------------------------------
def pair_f64(pi, pj, box, r):
    """O1-64 on one pair: returns (is_neighbor, d2_fp64)."""
    pi = np.ascontiguousarray(pi, np.float64)
    pj = np.ascontiguousarray(pj, np.float64)
    box = np.ascontiguousarray(box, np.float64)
    d2 = C.c_double()
    ok = lib().oracle_pair_f64(_p(pi, C.c_double), _p(pj, C.c_double), _p(box, C.c_double), C.c_double(float(r)), C.byref(d2))
    return bool(ok), float(d2.value)


def neighbor_list_f64(pos, type, box, r_list, method: str = "auto", timing: dict | None = None):
    """CSR neighbor list of fp64 positions by the definition in fp64.  Returns (row_ptr, nbr)."""
    pos = np.ascontiguousarray(pos, np.float64)
    N = pos.shape[0]
    assert pos.shape == (N, 3)
    type = None if type is None else np.ascontiguousarray(type, np.int32)
    box = np.ascontiguousarray(box, np.float64)
    r_list = np.ascontiguousarray(r_list, np.float64)
    T = r_list.shape[0]
    assert r_list.shape == (T, T)
    if method == "auto":
        method = "brute" if N <= 16384 else "cell"
    fn = {"brute": lib().oracle_brute_force_f64, "cell": lib().oracle_cell_list_f64}[method]
    t0 = time.perf_counter()
    n_neigh = np.zeros(max(N, 1), np.int32)
    args = [_p(pos, C.c_double), _p(type, C.c_int32), N, _p(box, C.c_double), _p(r_list, C.c_double), T]
    total = fn(*args, _p(n_neigh, C.c_int32), None, None)
    assert total >= 0
    row_ptr = np.zeros(N + 1, np.int64)
    np.cumsum(n_neigh[:N], out=row_ptr[1:])
    nbr = np.empty(max(int(total), 1), np.int32)
    total2 = fn(*args, _p(n_neigh, C.c_int32), _p(row_ptr, C.c_int64), _p(nbr, C.c_int32))
    assert total2 == total
    if timing is not None:
        timing["seconds"] = time.perf_counter() - t0
        timing["threads"] = num_threads()
        timing["method"] = method
    return row_ptr, nbr[:total]
