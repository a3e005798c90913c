"""fp64 brute-force CPU oracle for the SNAPS hot path -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` legs may import this package.  It does not import, and is
not imported by, paper_2405_20176_b200 (the CUDA path).  The arithmetic lives in
snaps_oracle.c (plain C, fp64, OpenMP over independent (mask, query) rows); this
file is the ctypes marshalling plus `build()`.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "snaps_oracle.c")
_LIB = os.path.join(_HERE, "libsnaps_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile snaps_oracle.c with gcc -O2 -fopenmp (no -ffast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.run(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                        "-o", tmp, _SRC, "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        c_i64, c_int = ctypes.c_int64, ctypes.c_int
        P = ctypes.c_void_p
        lib.snaps_oracle_num_threads.restype = c_int
        lib.snaps_oracle_knn.argtypes = [P, c_i64, c_int, c_i64, P, c_int, c_int, P, c_i64, P, P]
        lib.snaps_oracle_knn_scores.argtypes = [c_i64, c_int, c_int, P, P, P, P, P]
        lib.snaps_oracle_range.argtypes = [P, c_i64, c_int, c_i64, P, c_int, P, P, c_i64, P, P, P]
        lib.snaps_oracle_dist_row.argtypes = [P, c_i64, c_int, c_i64, ctypes.c_uint16, c_i64, P]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().snaps_oracle_num_threads())


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _prep(X, masks):
    X = np.ascontiguousarray(X, dtype=np.float32)
    assert X.ndim == 2
    masks = np.ascontiguousarray(masks, dtype=np.uint16).ravel()
    return X, masks


def _check(rc, what):
    if rc != 0:
        raise ValueError(f"oracle {what}: status {rc}")


def knn_selfjoin(X, masks, k, queries=None):
    """-> (idx int32 [n_masks][nq][k], dist fp64 same shape).  PAPER.md:112, 122."""
    X, masks = _prep(X, masks)
    N, n_feat = X.shape
    q = None if queries is None else np.ascontiguousarray(queries, dtype=np.int64)
    nq = N if q is None else len(q)
    idx = np.empty((len(masks), nq, k), dtype=np.int32)
    dist = np.empty((len(masks), nq, k), dtype=np.float64)
    _check(_load().snaps_oracle_knn(_ptr(X), N, n_feat, n_feat, _ptr(masks), len(masks), k,
                                    _ptr(q), nq, _ptr(idx), _ptr(dist)), "knn")
    return idx, dist


def knn_scores(N, idx, dist):
    """-> (kth, mean, indeg) each [n_masks][N].  PAPER.md:251-252; BASELINE.json configs[0]."""
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    dist = np.ascontiguousarray(dist, dtype=np.float64)
    n_masks, nq, k = idx.shape
    assert nq == N
    kth = np.empty((n_masks, N), dtype=np.float64)
    mean = np.empty((n_masks, N), dtype=np.float64)
    indeg = np.empty((n_masks, N), dtype=np.int64)
    _check(_load().snaps_oracle_knn_scores(N, n_masks, k, _ptr(idx), _ptr(dist),
                                           _ptr(kth), _ptr(mean), _ptr(indeg)), "knn_scores")
    return kth, mean, indeg


def range_selfjoin(X, masks, eps, queries=None):
    """-> (cnt int64, sum fp64, mean fp64) each [n_masks][nq].  PAPER.md:111, 156, 164-165."""
    X, masks = _prep(X, masks)
    N, n_feat = X.shape
    eps = np.ascontiguousarray(eps, dtype=np.float64).ravel()
    assert len(eps) == len(masks)
    q = None if queries is None else np.ascontiguousarray(queries, dtype=np.int64)
    nq = N if q is None else len(q)
    cnt = np.empty((len(masks), nq), dtype=np.int64)
    s = np.empty((len(masks), nq), dtype=np.float64)
    mean = np.empty((len(masks), nq), dtype=np.float64)
    _check(_load().snaps_oracle_range(_ptr(X), N, n_feat, n_feat, _ptr(masks), len(masks),
                                      _ptr(eps), _ptr(q), nq, _ptr(cnt), _ptr(s), _ptr(mean)),
           "range")
    return cnt, s, mean


def dist_row(X, mask, i):
    """All D(i, j; mask) for one query, fp64 [N]."""
    X = np.ascontiguousarray(X, dtype=np.float32)
    N, n_feat = X.shape
    out = np.empty(N, dtype=np.float64)
    _check(_load().snaps_oracle_dist_row(_ptr(X), N, n_feat, n_feat, int(mask), int(i), _ptr(out)),
           "dist_row")
    return out
