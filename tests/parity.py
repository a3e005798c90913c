"""Acceptance rules of BASELINE.json's north_star, shared by the GPU parity tests.

  kNN ids      equal to the oracle's as SETS for every query whose k-th -> (k+1)-th distance gap
               exceeds 1e-5 relative (reading A3); always: distinct, in range, never self
  kNN dists    within 1e-4 relative (absolute floor 1e-7), compared position by position on the
               ascending lists
  scores       kth / mean within 1e-4 relative; indeg == histogram of the GPU's own ids exactly,
               and == the oracle's where no query of that mask is ambiguous (reading A8)
  eps counts   cnt_oracle(eps(1-1e-6)) <= cnt_gpu <= cnt_oracle(eps(1+1e-6)) (reading A2)
"""
import numpy as np

RTOL = 1e-4
ATOL = 1e-7
GAP = 1e-5
BAND = 1e-6


def check_knn(gpu_idx, gpu_dist, or_idx_k1, or_dist_k1, queries=None):
    """gpu_*: [n_masks][nq][k]; or_*_k1: oracle run with k+1 neighbours."""
    gpu_idx = np.asarray(gpu_idx)
    gpu_dist = np.asarray(gpu_dist, dtype=np.float64)
    n_masks, nq, k = gpu_idx.shape
    or_idx, or_dist = or_idx_k1[:, :, :k], or_dist_k1[:, :, :k]
    q = np.arange(nq) if queries is None else np.asarray(queries)
    # validity, everywhere
    assert (gpu_idx >= 0).all()
    assert (gpu_idx != q[None, :, None]).all(), "self listed as a neighbour"
    srt = np.sort(gpu_idx, axis=2)
    assert (np.diff(srt, axis=2) > 0).all(), "duplicate neighbour ids"
    assert (np.diff(gpu_dist, axis=2) >= 0).all(), "distances not ascending"
    # distances
    err = np.abs(gpu_dist - or_dist)
    tol = RTOL * or_dist + ATOL
    assert (err <= tol).all(), f"distance mismatch: max rel {np.max(err / np.maximum(or_dist, 1e-30)):.3e}"
    # id sets where unambiguous
    dk, dk1 = or_dist_k1[:, :, k - 1], or_dist_k1[:, :, k]
    unamb = (dk1 - dk) > GAP * dk1
    same = (srt == np.sort(or_idx, axis=2)).all(axis=2)
    assert same[unamb].all(), f"{(~same & unamb).sum()} unambiguous id sets differ"
    # exact order where all consecutive gaps are unambiguous
    gaps = np.diff(or_dist_k1, axis=2) > GAP * or_dist_k1[:, :, 1:]
    strict = gaps.all(axis=2)
    assert (gpu_idx[strict] == or_idx[strict]).all()
    return unamb


def check_knn_scores(gpu, gpu_idx, or_kth, or_mean, or_indeg, unamb, N):
    kth = np.asarray(gpu["kth"], dtype=np.float64)
    mean = np.asarray(gpu["mean"], dtype=np.float64)
    indeg = np.asarray(gpu["indeg"])
    assert (np.abs(kth - or_kth) <= RTOL * or_kth + ATOL).all()
    assert (np.abs(mean - or_mean) <= RTOL * or_mean + ATOL).all()
    n_masks = indeg.shape[0]
    for m in range(n_masks):
        hist = np.bincount(np.asarray(gpu_idx[m]).ravel(), minlength=N)
        assert (indeg[m] == hist).all(), "in-degree is not the histogram of the GPU's ids"
        if unamb[m].all():
            assert (indeg[m] == or_indeg[m]).all()
    assert (indeg.sum(axis=1) == gpu_idx.shape[1] * gpu_idx.shape[2]).all()


def check_range(gpu_cnt, gpu_sum, gpu_mean, oracle_mod, X, masks, eps, queries=None):
    eps = np.asarray(eps, dtype=np.float32).astype(np.float64)   # what the GPU was given
    lo, s_lo, _ = oracle_mod.range_selfjoin(X, masks, eps * (1 - BAND), queries=queries)
    hi, s_hi, _ = oracle_mod.range_selfjoin(X, masks, eps * (1 + BAND), queries=queries)
    cnt = np.asarray(gpu_cnt).astype(np.int64)
    assert (lo <= cnt).all() and (cnt <= hi).all(), "eps-count outside the 1e-6 band"
    if gpu_sum is not None:
        s = np.asarray(gpu_sum, dtype=np.float64)
        assert (s >= s_lo * (1 - RTOL) - ATOL).all() and (s <= s_hi * (1 + RTOL) + ATOL).all()
    if gpu_mean is not None:
        mu = np.asarray(gpu_mean, dtype=np.float64)
        assert (mu[cnt == 0] == 0).all()                       # reading A6
        exact = lo == hi
        ref = np.where(lo > 0, s_lo / np.maximum(lo, 1), 0.0)
        assert (np.abs(mu - ref)[exact] <= RTOL * ref[exact] + ATOL).all()
    return lo, hi
