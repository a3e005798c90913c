"""Ranking, top-n overlap and parameter selection -- TEST INFRASTRUCTURE (oracle side, NEXT-1).

Plain numpy statements of PAPER.md section 3.4 (ranking function R), section 3.5.1 /
3.6.1 (which end of each metric is outlying), Eq. 2 (top-n overlap
f), Eq. 3 (parameter selection) and the nested-result rule
for the k grid (the neighbours for k_max contain those of every k_j < k_max).

Readings: ranks are DENSE and start at 0 = most outlying, ties share a rank
(verified on Table 2); an object with no eps-neighbour has mean distance 0 and
rank 0 in the distance-aware DSSJ metric; "top-n" = the first n objects of the
stable sort by (outlyingness, id) (reading A15: with shared ranks "r_i < n" would select more
than n objects); Eq. 3 takes the first index that attains the minimum.

Pins (tests/test_oracle_ranking.py): Table 2's four rank columns from its four metric columns;
the section 3.5.2 worked example (U_min = {1.0, 0.4, 0.2}, U_max = {0.2, 0.5, 1.0}).
"""
from __future__ import annotations

import numpy as np

# metric -> True if SMALL values are outlying (fewest neighbours / lowest in-degree),
# False if LARGE values are outlying (largest mean distance)
SMALL_IS_OUTLYING = {"dssj_count": True, "knn_indegree": True, "dssj_mean": False, "knn_mean": False,
                     "knn_kth": False}


def outlyingness_key(metric: str, values, counts=None) -> np.ndarray:
    """A float64 key that sorts most-outlying first (ascending).  For the distance-aware DSSJ
    metric, objects without neighbours (count 0) come before everything else."""
    v = np.asarray(values, dtype=np.float64)
    key = v.copy() if SMALL_IS_OUTLYING[metric] else -v
    if metric == "dssj_mean":
        assert counts is not None
        key = np.where(np.asarray(counts) == 0, -np.inf, key)
    return key


def dense_rank(metric: str, values, counts=None) -> np.ndarray:
    """R: rank 0 = most outlying; equal keys share a rank; ranks are consecutive."""
    key = outlyingness_key(metric, values, counts)
    uniq = np.unique(key)                      # ascending distinct keys
    return np.searchsorted(uniq, key).astype(np.int64)


def topn_ids(metric: str, values, n: int, counts=None) -> np.ndarray:
    """The n most outlying object ids: stable sort by (key, id) (reading A15)."""
    key = outlyingness_key(metric, values, counts)
    order = np.lexsort((np.arange(len(key)), key))
    return order[:n]


def overlap_fraction(ids_a, ids_b, n: int) -> float:
    """Eq. 2: f = |R^A ∩ R^B| / n over the two top-n sets."""
    return len(set(np.asarray(ids_a).tolist()) & set(np.asarray(ids_b).tolist())) / float(n)


def similarity_curves(topn_sets, n: int):
    """U_min[j] = f(top-n of grid point 0, of grid point j); U_max[j] = f(last, j)."""
    g = len(topn_sets)
    u_min = np.array([overlap_fraction(topn_sets[0], topn_sets[j], n) for j in range(g)])
    u_max = np.array([overlap_fraction(topn_sets[g - 1], topn_sets[j], n) for j in range(g)])
    return u_min, u_max


def select_parameter(u_min, u_max, n: int | None = None) -> int:
    """Eq. 3: argmin_j |U_min[j] - U_max[j]| (first minimiser).  With n given the
    fractions are taken back to their integer hit counts first, so that equal differences are
    exactly equal (f = hits / n: ties must not be decided by floating-point rounding)."""
    a, b = np.asarray(u_min, dtype=np.float64), np.asarray(u_max, dtype=np.float64)
    if n is not None:
        a, b = np.rint(a * n), np.rint(b * n)
    return int(np.argmin(np.abs(a - b)))


def knn_scores_at_k(idx_kmax, dist_kmax, kj: int, N: int):
    """Scores for k_j from the k_max lists: the first k_j columns.
    idx/dist: [N][k_max] of one mask.  -> (kth, mean, indeg)."""
    idx = np.asarray(idx_kmax)[:, :kj]
    dist = np.asarray(dist_kmax, dtype=np.float64)[:, :kj]
    return dist[:, -1], dist.mean(axis=1), np.bincount(idx.ravel(), minlength=N)


def mean_in_list_order_fp32(dist_kmax, kj: int) -> np.ndarray:
    """The mean kNN distance as a 32-bit value: the first k_j distances added one by one in list order
    in fp32, then divided by k_j ("32-bit floating point" throughout).  Rank decisions on
    the distance-aware kNN metric are taken on this value (reading A21), so that objects whose
    means differ by less than an fp32 rounding do not change order between implementations."""
    d = np.asarray(dist_kmax, dtype=np.float32)[:, :kj]
    return (np.cumsum(d, axis=1, dtype=np.float32)[:, -1] / np.float32(kj)).astype(np.float32)


def select_k(idx_kmax, dist_kmax, k_grid, n: int, N: int):
    """The k-grid procedure of PAPER.md:256-258 for ONE mask, step by step: for every k_j the scores
    from the k_max lists, their top-n sets, U_min / U_max against the smallest and largest k
    (Eq. 2), and the selected grid index (Eq. 3) -- for the in-degree and the mean-distance metric.
    The mean-distance ranks are decided on the fp32 mean (reading A21).
    -> dict metric -> (j_select, u_min, u_max)."""
    out = {}
    for metric, pick in (("knn_indegree", 2), ("knn_mean", 1)):
        tops = []
        for kj in k_grid:
            sc = knn_scores_at_k(idx_kmax, dist_kmax, int(kj), N)
            score = sc[pick] if metric == "knn_indegree" else mean_in_list_order_fp32(dist_kmax, int(kj))
            tops.append(topn_ids(metric, score, n))
        u_min, u_max = similarity_curves(tops, n)
        out[metric] = (select_parameter(u_min, u_max, n), u_min, u_max)
    return out


def eps_grid(eps_min, eps_max, G: int) -> np.ndarray:
    """The grid G of PAPER.md:181: |G| evenly spaced radii, eps_1 = eps_min, eps_|G| = eps_max
    (PAPER.md:183), carried as 32-bit values with every operation rounded:
    eps_j = eps_min + (j - 1) * ((eps_max - eps_min) / (|G| - 1)), the last one eps_max itself."""
    e0, e1 = np.float32(eps_min), np.float32(eps_max)
    step = np.float32(np.float32(e1 - e0) / np.float32(G - 1))
    grid = np.array([np.float32(e0 + np.float32(np.float32(g) * step)) for g in range(G)], dtype=np.float32)
    grid[G - 1] = e1
    return grid


def select_eps(counts, means, n: int):
    """The eps-grid procedure of PAPER.md:181-189 for ONE mask from the join results at every radius
    (counts [G][N], means [G][N]; means 0 where the count is 0): top-n sets per radius for the number-of-
    neighbours metric and the mean-distance metric, U_min / U_max against the smallest and the largest
    radius (Eq. 2), the selected grid index (Eq. 3).  -> dict metric -> (j_select, u_min, u_max)."""
    out = {}
    G = len(counts)
    tops = [topn_ids("dssj_count", counts[g], n) for g in range(G)]
    u_min, u_max = similarity_curves(tops, n)
    out["dssj_count"] = (select_parameter(u_min, u_max, n), u_min, u_max)
    tops = [topn_ids("dssj_mean", means[g], n, counts=counts[g]) for g in range(G)]
    u_min, u_max = similarity_curves(tops, n)
    out["dssj_mean"] = (select_parameter(u_min, u_max, n), u_min, u_max)
    return out


def range_from_knn(dist_k, eps: float):
    """kNN -> DSSJ reuse for ONE mask, from the definitions: with the k nearest neighbours of
    every object sorted by distance, the objects within eps are a prefix of the list; if the k-th neighbour
    lies beyond eps the prefix is the whole eps-neighbourhood.
    dist_k: [N][k] ascending.  -> (count, sumdist, mean, complete)."""
    d = np.asarray(dist_k)
    inside = d <= d.dtype.type(eps)
    cnt = inside.sum(axis=1)
    s = np.where(inside, d, 0).sum(axis=1, dtype=np.float64)
    mean = np.where(cnt > 0, s / np.maximum(cnt, 1), 0.0)
    return cnt, s, mean, cnt < d.shape[1]
