"""Pins for the fp64 oracle against what the paper and the mathematics fix
(SURVEY.md 8(c) "What pins each part"): closed forms, a library routine,
exhaustive enumeration, invariants.  None of these re-types the oracle's loop."""
import itertools
import math
import os

import numpy as np
import pytest
from scipy.spatial import cKDTree
from scipy.special import comb

import workloads

HERE = os.path.dirname(os.path.abspath(__file__))


# ---------------------------------------------------------------- Eq. 1
def test_eq1_mask_count():
    # PAPER.md:142 Eq. 1: sum_{i=2}^{15} C(15,i) = 32,752
    m = workloads.all_masks(15)
    assert len(m) == 32752 == (1 << 15) - 1 - 15
    assert len(set(m.tolist())) == 32752
    assert (workloads.popcount(m) >= 2).all()
    assert len(workloads.all_masks(4)) == 11  # BASELINE.json configs[0]
    assert len(workloads.pair_masks_plus_full(15)) == 106


def test_table2_internal_consistency():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "table2_paper.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 10
    assert sum(int(r[5]) for r in rows) == 30          # N*k directed edges
    assert sum(int(r[1]) for r in rows) % 2 == 0       # symmetric eps-join
    assert all(float(r[3]) <= 0.67 for r in rows)      # mean of distances <= eps
    assert [r for r in rows if int(r[1]) == 0][0][3] == "0.0000"  # reading A6


# ---------------------------------------------------------------- distance closed forms
def test_one_feature_and_duplicated_column(oracle_mod):
    rng = np.random.default_rng(5)
    X = rng.random((40, 4)).astype(np.float32)
    X[:, 2] = X[:, 1]                                   # column 2 := column 1
    for i in (0, 7, 39):
        d1 = oracle_mod.dist_row(X, 0b0010, i)
        np.testing.assert_allclose(d1, np.abs(X[:, 1].astype(np.float64) - float(X[i, 1])), rtol=1e-15)
        d2 = oracle_mod.dist_row(X, 0b0110, i)
        np.testing.assert_allclose(d2, math.sqrt(2.0) * d1, rtol=1e-15)
        # a transposed operand / wrong column would break this one
        d3 = oracle_mod.dist_row(X, 0b1001, i)
        ref = np.hypot(X[:, 0].astype(np.float64) - float(X[i, 0]), X[:, 3].astype(np.float64) - float(X[i, 3]))
        np.testing.assert_allclose(d3, ref, rtol=1e-15)


def test_power_of_two_scaling_is_exact(oracle_mod):
    rng = np.random.default_rng(6)
    X = rng.random((30, 3)).astype(np.float32)
    idx_a, d_a = oracle_mod.knn_selfjoin(X, [0b111], 4)
    idx_b, d_b = oracle_mod.knn_selfjoin(X * np.float32(0.25), [0b111], 4)
    assert (idx_a == idx_b).all()
    assert (d_b == 0.25 * d_a).all()


# ---------------------------------------------------------------- 1-D lattice (closed form A)
def test_lattice_closed_form(oracle_mod):
    n, h, k = 64, 2.0 ** -7, 6
    X = workloads.lattice_table(n, 3, h, seed=1)
    idx, dist = oracle_mod.knn_selfjoin(X, [0b001], k)
    kth, mean, indeg = oracle_mod.knn_scores(n, idx, dist)
    for i in range(n):
        # distances to the others are |i-j|*h; ties (i-r, i+r) go to the smaller id
        others = sorted((abs(i - j) * h, j) for j in range(n) if j != i)[:k]
        assert idx[0, i].tolist() == [j for _, j in others]
        assert dist[0, i].tolist() == [d for d, _ in others]
    # in-degree: object j counts the queries i whose list holds j.  Closed form on
    # the lattice from the id lists derived above (NOT from the oracle's own idx): interior
    # objects are listed by their k nearest lattice sites (k), the sites near a boundary also by
    # the boundary queries whose lists are one-sided -- in-degree != out-degree there.
    exp_indeg = np.zeros(n, dtype=np.int64)
    for i in range(n):
        for _, j in sorted((abs(i - j) * h, j) for j in range(n) if j != i)[:k]:
            exp_indeg[j] += 1
    assert indeg[0].tolist() == exp_indeg.tolist()
    # written out: site j <= k is listed by k/2 + j queries (the one-sided lists of the first k/2
    # queries pile up on sites 0..k), sites k < j < n-1-k by exactly k, mirrored at the far end
    closed = np.full(n, k)
    closed[:k + 1] = k // 2 + np.arange(k + 1)
    closed[n - k - 1:] = (k // 2 + np.arange(k + 1))[::-1]
    assert indeg[0].tolist() == closed.tolist()
    interior = np.arange(k // 2, n - k // 2)
    assert (kth[0, interior] == (k // 2) * h).all()
    np.testing.assert_allclose(mean[0, interior], h * (k / 2 + 1) / 2, rtol=1e-15)
    assert kth[0, 0] == k * h and mean[0, 0] == h * (k + 1) / 2          # boundary point
    cnt, s, mu = oracle_mod.range_selfjoin(X, [0b001], [2.5 * h])
    assert (cnt[0, 2:-2] == 4).all() and cnt[0, 0] == 2 and cnt[0, 1] == 3
    np.testing.assert_allclose(s[0, 2:-2], 6 * h, rtol=1e-15)
    # closed ball (reading A2): eps exactly on a lattice distance includes it
    cnt2, _, _ = oracle_mod.range_selfjoin(X, [0b001], [2.0 * h])
    assert (cnt2[0, 2:-2] == 4).all()


def test_indegree_asymmetric_hand_example(oracle_mod):
    # Four collinear objects at x = 0, 1, 2, 10 (scaled into [0,1]), k = 1.  Nearest neighbours by
    # hand: 0 -> 1, 1 -> 0 (tie |1-0| = |1-2| goes to the smaller id, reading A3), 2 -> 1, 3 -> 2.
    # In-degree ("number of occurrences that a point is found within another point's
    # set of kNN") = {1, 2, 1, 0}: differs from the out-degree k = 1 of every object, so an
    # accumulation at the query index instead of the neighbour id cannot pass.  Table 2's own
    # in-degree column (5,6,6,3,2,3,2,2,1,0 for k = 3) shows the same asymmetry.
    X = (np.array([[0.0], [1.0], [2.0], [10.0]]) / 16.0).astype(np.float32)
    idx, dist = oracle_mod.knn_selfjoin(X, [0b1], 1)
    assert idx[0, :, 0].tolist() == [1, 0, 1, 2]
    kth, mean, indeg = oracle_mod.knn_scores(4, idx, dist)
    assert indeg[0].tolist() == [1, 2, 1, 0]
    assert kth[0].tolist() == [1 / 16, 1 / 16, 1 / 16, 8 / 16]
    # k = 2: 0 -> {1,2}, 1 -> {0,2}, 2 -> {1,0}, 3 -> {2,1}
    idx2, dist2 = oracle_mod.knn_selfjoin(X, [0b1], 2)
    assert idx2[0].tolist() == [[1, 2], [0, 2], [1, 0], [2, 1]]
    _, mean2, indeg2 = oracle_mod.knn_scores(4, idx2, dist2)
    assert indeg2[0].tolist() == [2, 3, 3, 0]
    assert mean2[0].tolist() == [1.5 / 16, 1 / 16, 1.5 / 16, 8.5 / 16]
    # the k-grid helper of the ranking oracle reads the same lists
    from oracle import ranking
    _, _, g1 = ranking.knn_scores_at_k(idx2[0], dist2[0], 1, 4)
    _, _, g2 = ranking.knn_scores_at_k(idx2[0], dist2[0], 2, 4)
    assert g1.tolist() == [1, 2, 1, 0] and g2.tolist() == [2, 3, 3, 0]


# ---------------------------------------------------------------- hypercube (closed form B, ties)
@pytest.mark.parametrize("nf", [6, 9])
def test_hypercube_counts_and_order_statistics(oracle_mod, nf):
    X = workloads.hypercube_table(nf)
    n = 1 << nf
    rng = np.random.default_rng(nf)
    masks = rng.choice(workloads.all_masks(nf, 1), 6, replace=False)
    for eps in (0.5, 1.0, 1.5, 2.01):
        cnt, s, mu = oracle_mod.range_selfjoin(X, masks, np.full(len(masks), eps))
        for mi, m in enumerate(masks):
            d = bin(int(m)).count("1")
            mult = 1 << (nf - d)
            exp_cnt = sum(comb(d, r, exact=True) * mult for r in range(d + 1) if math.sqrt(r) <= eps) - 1
            exp_sum = sum(comb(d, r, exact=True) * mult * math.sqrt(r) for r in range(d + 1) if math.sqrt(r) <= eps)
            assert (cnt[mi] == exp_cnt).all()
            np.testing.assert_allclose(s[mi], exp_sum, rtol=1e-12)
            np.testing.assert_allclose(mu[mi], exp_sum / exp_cnt if exp_cnt else 0.0, rtol=1e-12)
    k = 10
    idx, dist = oracle_mod.knn_selfjoin(X, masks, k)
    for mi, m in enumerate(masks):
        d = bin(int(m)).count("1")
        mult = 1 << (nf - d)
        levels = []                                    # sorted distance multiset of any vertex
        for r in range(d + 1):
            levels += [math.sqrt(r)] * (comb(d, r, exact=True) * mult - (1 if r == 0 else 0))
        assert (dist[mi] == np.array(levels[:k])).all()
        assert (idx[mi] != np.arange(n)[:, None]).all()  # self excluded by index (A4)
        # tie-break to smaller id (A3): zero-distance twins are listed first, ascending id
        n_zero = min(k, mult - 1)
        if n_zero:
            twins = np.sort(idx[mi][:, :n_zero], axis=1)
            assert (twins == idx[mi][:, :n_zero]).all()


# ---------------------------------------------------------------- library routine (scipy cKDTree)
@pytest.mark.parametrize("seed,n,nf", [(0, 300, 5), (1, 257, 15)])
def test_against_ckdtree(oracle_mod, seed, n, nf):
    X = workloads.make_table(n, seed, cols=list(range(nf)))
    rng = np.random.default_rng(seed)
    masks = rng.choice(workloads.all_masks(nf), 5, replace=False)
    k = 7
    idx, dist = oracle_mod.knn_selfjoin(X, masks, k)
    eps = np.array([np.median(dist[mi, :, -1]) for mi in range(len(masks))])
    cnt, s, mu = oracle_mod.range_selfjoin(X, masks, eps)
    for mi, m in enumerate(masks):
        cols = [f for f in range(nf) if (int(m) >> f) & 1]
        sub = X[:, cols].astype(np.float64)
        tree = cKDTree(sub)
        dd, ii = tree.query(sub, k=k + 1)
        # continuous data: no exact ties, self is the 0-distance hit in column 0
        assert (ii[:, 0] == np.arange(n)).all()
        assert (idx[mi] == ii[:, 1:]).all()
        np.testing.assert_allclose(dist[mi], dd[:, 1:], rtol=1e-12)
        balls = tree.query_ball_point(sub, eps[mi] * (1 + 1e-12))
        lib_cnt = np.array([len(b) - 1 for b in balls])
        assert (cnt[mi] == lib_cnt).all()
        lib_sum = np.array([np.linalg.norm(sub[b] - sub[i], axis=1).sum() for i, b in enumerate(balls)])
        np.testing.assert_allclose(s[mi], lib_sum, rtol=1e-10, atol=1e-14)


# ---------------------------------------------------------------- exhaustive, tiny N
def test_knn_exhaustive_enumeration(oracle_mod):
    rng = np.random.default_rng(11)
    for trial in range(5):
        n = int(rng.integers(4, 9))
        X = np.round(rng.random((n, 3)) * 4).astype(np.float32) / 4      # coarse grid => ties
        for k in (1, 2, 3):
            for m in (0b001, 0b011, 0b111, 0b110):
                idx, dist = oracle_mod.knn_selfjoin(X, [m], k)
                cols = [f for f in range(3) if (m >> f) & 1]
                for i in range(n):
                    others = [j for j in range(n) if j != i]
                    best = None
                    for sub in itertools.combinations(others, k):
                        key = sorted((float(np.sqrt(((X[i, cols].astype(np.float64) - X[j, cols]) ** 2).sum())), j)
                                     for j in sub)
                        if best is None or key < best:
                            best = key
                    assert [j for _, j in best] == idx[0, i].tolist()
                    np.testing.assert_allclose([d for d, _ in best], dist[0, i], rtol=1e-15)


# ---------------------------------------------------------------- invariants
def test_invariants_on_config1(oracle_mod):
    cfg = workloads.get_config("c1_tiny")
    X, masks, k = cfg.table(), cfg.masks(), cfg.k
    n = len(X)
    idx, dist = oracle_mod.knn_selfjoin(X, masks, k)
    kth, mean, indeg = oracle_mod.knn_scores(n, idx, dist)
    assert (indeg.sum(axis=1) == n * k).all()
    assert (np.diff(dist, axis=2) >= 0).all()
    assert (mean <= kth + 1e-15).all()
    assert (idx != np.arange(n)[None, :, None]).all()
    assert all(len(set(r)) == k for r in idx.reshape(-1, k).tolist())
    # order statistics are monotone along lattice edges S -> S u {f}
    pos = {int(m): i for i, m in enumerate(masks)}
    for m in masks:
        for f in range(4):
            if not (int(m) >> f) & 1 and (int(m) | (1 << f)) in pos:
                assert (dist[pos[int(m)]] <= dist[pos[int(m) | (1 << f)]] + 1e-15).all()
    # eps-join: symmetric, nested in eps, consistent with kNN ranks
    eps = np.array([np.median(kth[mi]) for mi in range(len(masks))])
    cnt, s, mu = oracle_mod.range_selfjoin(X, masks, eps)
    cnt_small, _, _ = oracle_mod.range_selfjoin(X, masks, 0.5 * eps)
    assert (cnt.sum(axis=1) % 2 == 0).all()                          # pair (i,j) <=> (j,i)
    assert (cnt_small <= cnt).all()                                  # PAPER.md:235 Fig. 3 nesting
    for m in masks:
        for f in range(4):
            if not (int(m) >> f) & 1 and (int(m) | (1 << f)) in pos:
                a, b = pos[int(m)], pos[int(m) | (1 << f)]
                c_sup, _, _ = oracle_mod.range_selfjoin(X, [masks[b]], [eps[a]])
                assert (c_sup[0] <= cnt[a]).all()
    for mi in (0, 5, 10):
        for i in (0, 17, 1999):
            c_at, _, _ = oracle_mod.range_selfjoin(X, [masks[mi]], [kth[mi, i]], queries=[i])
            assert c_at[0, 0] >= k
            c_below, _, _ = oracle_mod.range_selfjoin(X, [masks[mi]], [kth[mi, i] * (1 - 1e-12)], queries=[i])
            assert c_below[0, 0] <= k - 1 or kth[mi, i] == 0.0
    assert (mu[cnt == 0] == 0).all() and (s[cnt == 0] == 0).all()


def test_permutation_equivariance(oracle_mod):
    X = workloads.make_table(200, 9, cols=[0, 1, 2, 3, 4])
    masks = np.array([0b00110, 0b11001, 0b11111], dtype=np.uint16)
    idx, dist = oracle_mod.knn_selfjoin(X, masks, 5)
    rng = np.random.default_rng(3)
    perm = rng.permutation(200)
    idx_p, dist_p = oracle_mod.knn_selfjoin(X[perm], masks, 5)
    np.testing.assert_array_equal(dist_p, dist[:, perm])
    assert (perm[idx_p] == idx[:, perm]).all()
    cperm = np.array([3, 0, 4, 1, 2])                     # new column c holds old column cperm[c]
    masks_p = np.array([sum(1 << c for c in range(5) if (int(m) >> cperm[c]) & 1) for m in masks], dtype=np.uint16)
    idx_c, dist_c = oracle_mod.knn_selfjoin(X[:, cperm], masks_p, 5)
    assert (idx_c == idx).all()
    np.testing.assert_allclose(dist_c, dist, rtol=1e-14)


def test_sampled_queries_equal_full_rows(oracle_mod):
    X = workloads.make_table(150, 2, cols=[0, 1, 2])
    masks = workloads.all_masks(3)
    idx, dist = oracle_mod.knn_selfjoin(X, masks, 4)
    q = np.array([149, 3, 77])
    idx_q, dist_q = oracle_mod.knn_selfjoin(X, masks, 4, queries=q)
    assert (idx_q == idx[:, q]).all() and (dist_q == dist[:, q]).all()


def test_duplicate_block_self_exclusion(oracle_mod):
    # reading A4/A7: a different object at distance 0 is a neighbour; self never is
    X = workloads.duplicate_block_table(400, 3, frac=0.3)
    m = np.array([(1 << 13) | (1 << 14)], dtype=np.uint16)
    idx, dist = oracle_mod.knn_selfjoin(X, m, 8)
    vals, counts = np.unique(X[:, 13], return_counts=True)
    block_val = vals[np.argmax(counts)]
    block = np.flatnonzero((X[:, 13] == block_val) & (X[:, 14] == X[np.argmax(X[:, 13] == block_val), 14]))
    assert len(block) >= 100
    assert (dist[0, block] == 0).all()
    assert (idx[0, block] != block[:, None]).all()
    # smallest ids of the block, skipping self
    for i in block[:5]:
        assert idx[0, i].tolist() == [j for j in block.tolist() if j != i][:8]


def test_oracle_rejects_bad_arguments(oracle_mod):
    X = np.zeros((5, 3), dtype=np.float32)
    with pytest.raises(ValueError):
        oracle_mod.knn_selfjoin(X, [0b111], 5)            # k <= N-1 (A9)
    with pytest.raises(ValueError):
        oracle_mod.knn_selfjoin(X, [0], 2)                # empty mask
    with pytest.raises(ValueError):
        oracle_mod.knn_selfjoin(X, [0b1000], 2)           # bit >= n_feat
    with pytest.raises(ValueError):
        oracle_mod.range_selfjoin(X, [0b1], [0.0])        # eps > 0


# ---------------------------------------------------------------- NEXT-2: sampled distance histogram
def test_sampled_histogram_closed_form_and_selectivity(oracle_mod):
    from oracle.calibrate import sampled_histogram, eps_from_histogram
    n, h = 64, 2.0 ** -7
    X = workloads.lattice_table(n, 3, h, seed=2)
    ids = np.arange(n)
    # 1-D lattice, all points sampled: |i-j| h for i != j -> 2 (n - r) ordered pairs at distance r h
    hist, _ = sampled_histogram(X, [0b001], ids, ids, [n * h], n)          # bin width = h, bin r holds r h
    assert hist[0, 0] == 0 and all(hist[0, r] == 2 * (n - r) for r in range(1, n))
    # with every object sampled the cumulative histogram IS the eps-join: sum of counts at radius
    # just below a bin edge (open bins, closed ball: keep eps off the lattice distances)
    cnt, _, _ = oracle_mod.range_selfjoin(X, [0b001], [4.5 * h])
    assert hist[0, :5].sum() == cnt[0].sum()
    # selectivity: mean neighbours = cum * (N-1) / pairs; target 6 -> first edge reaching it
    eps = eps_from_histogram(hist, [n * h], n, n * (n - 1), 6.0)
    mean_at = lambda r: oracle_mod.range_selfjoin(X, [0b001], [r])[0].mean()
    assert mean_at(eps[0] * (1 - 1e-9)) >= 6.0 > mean_at((eps[0] - h) * (1 - 1e-9))


def test_eps_search_lattice_closed_forms(oracle_mod):
    """eps_mean and the radii of oracle.calibrate.eps_search on the 1-D lattice with every object sampled:
    the mean of |i - j| h over i != j is (n + 1) h / 3; the radius for a target of s neighbours is the
    first bin edge whose ball holds them."""
    from oracle.calibrate import eps_search, mean_sample_distance
    n, h = 48, 2.0 ** -8
    X = workloads.lattice_table(n, 3, h, seed=4)
    ids = np.arange(n)
    em, pairs = mean_sample_distance(X, [0b001], ids, ids)
    assert pairs == n * (n - 1) and abs(em[0] - (n + 1) * h / 3) < 1e-15
    # a two-feature mask with a duplicated column scales every distance by sqrt(2)
    X2 = X.copy()
    X2[:, 1] = X2[:, 0]
    em2, _ = mean_sample_distance(X2, [0b011], ids, ids)
    assert abs(em2[0] / em[0] - np.sqrt(2.0)) < 1e-12
    rmax, eps, hist, _ = eps_search(X, [0b001], ids, ids, 256, [2.0, 6.0])
    assert rmax[0] == np.float32((n + 1) * h / 3) and hist[0].sum() <= pairs
    mean_at = lambda r: oracle_mod.range_selfjoin(X, [0b001], [r])[0].mean()
    w = float(rmax[0]) / 256
    for t, e in zip((2.0, 6.0), eps[0]):
        assert mean_at(float(e) * (1 - 1e-9)) >= t > mean_at((float(e) - w) * (1 - 1e-9))


def test_eps_grid_matches_figure_2(oracle_mod):
    """the example feature space of Fig. 2 has eps_min = 0.0360, eps_max = 0.1707 and its
    selected radius eps = 0.1256 is grid point arg = 15 (counted from 1).  With evenly spaced radii that
    fixes |G| = 22 (step 0.0064); the oracle's grid must put its 15th point there, up to the rounding of
    the published four-digit values.  (A division by |G| instead of |G| - 1, or an index off by one, misses
    by more than ten times that.)"""
    from oracle.ranking import eps_grid
    g = eps_grid(0.0360, 0.1707, 22)
    assert g[0] == np.float32(0.0360) and g[-1] == np.float32(0.1707) and len(g) == 22
    assert abs(float(g[14]) - 0.1256) < 3.5e-4
    assert abs(float(g[15]) - 0.1256) > 3e-3 and abs(float(g[13]) - 0.1256) > 3e-3
    assert np.allclose(np.diff(g.astype(np.float64)), (0.1707 - 0.0360) / 21, rtol=1e-5)
