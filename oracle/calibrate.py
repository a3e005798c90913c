"""eps_d calibration for the DSSJ configs -- TEST INFRASTRUCTURE (oracle side).

A reduced form of the paper's sampled cumulative distance histogram
(section 3.5.3): the radius at which a sample's pooled pair
distances reach the target selectivity s = mean neighbours per point
(PAPER.md:221).  Recipe in DESIGN.md "Input recipe".
"""
from __future__ import annotations

import numpy as np

from . import dist_row


def eps_per_dimension(X, masks, target_neighbours, seed, n_query_sample=1000,
                      n_cand_sample=None, max_masks_per_dim=64):
    """-> eps [n_masks] fp64: every mask of popcount d gets eps_d, the pooled
    sample quantile at target_neighbours/(N-1) of D over (sampled query,
    sampled candidate != query) pairs of up to max_masks_per_dim masks of that d."""
    X = np.ascontiguousarray(X, dtype=np.float32)
    masks = np.asarray(masks, dtype=np.uint16)
    N = X.shape[0]
    rng = np.random.default_rng(seed)
    qs = np.sort(rng.choice(N, min(n_query_sample, N), replace=False))
    if n_cand_sample is None or n_cand_sample >= N:
        cs = qs
    else:
        cs = np.sort(rng.choice(N, n_cand_sample, replace=False))
    Xs = np.ascontiguousarray(X[np.union1d(qs, cs)])
    ids = np.union1d(qs, cs)
    q_pos = np.searchsorted(ids, qs)
    c_pos = np.searchsorted(ids, cs)
    dims = np.array([bin(int(m)).count("1") for m in masks])
    frac = target_neighbours / (N - 1)
    eps = np.zeros(len(masks), dtype=np.float64)
    for d in np.unique(dims):
        sel = np.flatnonzero(dims == d)
        pick = sel if len(sel) <= max_masks_per_dim else np.sort(
            rng.permutation(sel)[:max_masks_per_dim])
        pooled = []
        for mi in pick:
            for qp in q_pos:
                row = dist_row(Xs, masks[mi], qp)[c_pos]
                keep = c_pos != qp
                pooled.append(row[keep])
        pooled = np.concatenate(pooled)
        eps[sel] = np.quantile(pooled, frac)
    return eps


def sampled_histogram(X, masks, q_ids, c_ids, rmax, n_bins: int):
    """NEXT-2 oracle: per mask the histogram of D(q, c; mask) over the sampled
    queries x sampled candidates (c != q by index), n_bins equal half-open bins [b w, (b+1) w) over
    [0, rmax); pairs at or beyond rmax are not counted.  fp64, one distance at a time.
    -> (hist int64 [n_masks][n_bins], distances list per mask for band checks)."""
    X = np.ascontiguousarray(X, dtype=np.float32)
    masks = np.asarray(masks, dtype=np.uint16)
    q_ids = np.asarray(q_ids, dtype=np.int64)
    c_ids = np.asarray(c_ids, dtype=np.int64)
    hist = np.zeros((len(masks), n_bins), dtype=np.int64)
    all_d = []
    for mi, m in enumerate(masks):
        ds = []
        for q in q_ids:
            row = dist_row(X, m, int(q))[c_ids]
            ds.append(row[c_ids != q])
        d = np.concatenate(ds)
        all_d.append(d)
        b = np.floor(d / float(rmax[mi]) * n_bins).astype(np.int64)
        hist[mi] = np.bincount(b[b < n_bins], minlength=n_bins)[:n_bins]
    return hist, all_d


def eps_from_histogram(hist, rmax, N: int, pairs_per_mask: int, target_s: float):
    """Cumulative histogram -> smallest bin edge whose mean neighbour count (selectivity s,
    PAPER.md:221) reaches target_s; rmax if none does."""
    hist = np.asarray(hist, dtype=np.float64)
    eps = np.array(rmax, dtype=np.float64).copy()
    for mi in range(hist.shape[0]):
        mean = np.cumsum(hist[mi]) * (N - 1) / float(pairs_per_mask)
        hit = np.flatnonzero(mean >= target_s)
        if len(hit):
            eps[mi] = float(rmax[mi]) * (hit[0] + 1) / hist.shape[1]
    return eps


def mean_sample_distance(X, masks, q_ids, c_ids):
    """eps_mean: the mean of D(q, c; mask) over the sampled (query, candidate) pairs with
    c != q by index -- "the mean distance between points in a dataset", estimated on a sample and used as
    the upper bound of the search radius.  fp64.  -> (eps_mean [n_masks], number of pairs)."""
    X = np.ascontiguousarray(X, dtype=np.float32)
    q_ids = np.asarray(q_ids, dtype=np.int64)
    c_ids = np.asarray(c_ids, dtype=np.int64)
    out = np.zeros(len(masks), dtype=np.float64)
    pairs = 0
    for mi, m in enumerate(masks):
        tot, cnt = 0.0, 0
        for q in q_ids:
            row = dist_row(X, m, int(q))[c_ids]
            keep = c_ids != q
            tot += float(row[keep].sum())
            cnt += int(keep.sum())
        out[mi] = tot / cnt
        pairs = cnt
    return out, pairs


def eps_search(X, masks, q_ids, c_ids, n_bins: int, targets):
    """The search of PAPER.md:229-237, step by step: eps_mean from the sample; the histogram of the sampled
    distances over [0, eps_mean) (the range as the 32-bit value the method carries); its
    cumulative form -> for every target selectivity the first bin edge that reaches it (eps_mean if none).
    -> (eps_mean fp32 [n_masks], eps fp32 [n_masks][n_targets], hist, distances per mask)."""
    N = len(X)
    eps_mean, pairs = mean_sample_distance(X, masks, q_ids, c_ids)
    rmax = eps_mean.astype(np.float32)
    hist, dists = sampled_histogram(X, masks, q_ids, c_ids, rmax, n_bins)
    eps = np.stack([eps_from_histogram(hist, rmax, N, pairs, float(t)) for t in targets], axis=1)
    return rmax, eps.astype(np.float32), hist, dists
