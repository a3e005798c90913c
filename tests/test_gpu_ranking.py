"""GPU parity for NEXT-1 (ranking, top-n overlap, parameter selection, k-grid scores) against
oracle/ranking.py -- integer / index work: bit-exact on the same score arrays."""
import os

import numpy as np
import pytest

import workloads
from oracle import ranking as oracle_ranking

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def snaps():
    import torch
    assert torch.cuda.is_available()
    import paper_2405_20176_b200 as s
    s.lib()
    return s


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_table2_ranks_on_device(snaps):
    import torch
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "table2_paper.txt"))
            if l.strip() and not l.startswith("#")]
    t = np.array(rows, dtype=np.float64)
    cnt = t[:, 1].astype(np.uint32)
    cases = [("dssj_count", cnt.view(np.int32), None, t[:, 2]),
             ("dssj_mean", t[:, 3].astype(np.float32), cnt.view(np.int32), t[:, 4]),
             ("knn_indegree", t[:, 5].astype(np.int32), None, t[:, 6]),
             ("knn_mean", t[:, 7].astype(np.float32), None, t[:, 8])]
    for metric, vals, counts, want in cases:
        out = snaps.rank_scores(metric, _t(vals[None, :]), None if counts is None else _t(counts[None, :]))
        torch.cuda.synchronize()
        assert out["rank"][0].cpu().numpy().tolist() == want.astype(int).tolist(), metric


@pytest.mark.parametrize("metric", ["dssj_count", "dssj_mean", "knn_indegree", "knn_mean"])
@pytest.mark.parametrize("n_rows,N", [(1, 1), (3, 257), (7, 5000), (2, 31693)])
def test_rank_and_order_match_oracle(snaps, metric, n_rows, N):
    import torch
    rng = np.random.default_rng(N + n_rows)
    counts = None
    if metric in ("dssj_count", "knn_indegree"):
        vals = rng.integers(0, max(2, N // 20), (n_rows, N)).astype(np.int32)      # many ties
    else:
        vals = np.round(rng.random((n_rows, N)) * 50).astype(np.float32) / 50        # ties too
        if metric == "dssj_mean":
            counts = rng.integers(0, 4, (n_rows, N)).astype(np.int32)
            vals[counts == 0] = 0.0                                                  # reading A6
    out = snaps.rank_scores(metric, _t(vals), None if counts is None else _t(counts))
    torch.cuda.synchronize()
    for r in range(n_rows):
        c = None if counts is None else counts[r]
        assert (out["rank"][r].cpu().numpy() == oracle_ranking.dense_rank(metric, vals[r], c)).all()
        assert (out["order"][r].cpu().numpy() == oracle_ranking.topn_ids(metric, vals[r], N, c)).all()


def test_overlap_and_selection_worked_example(snaps):
    # the section 3.5.2 example through the device kernels
    import torch
    rec = {}
    for l in open(os.path.join(HERE, "golden", "section352_example.txt")):
        if l.strip() and not l.startswith("#"):
            p = l.split()
            rec[p[0]] = [float(x) for x in p[1:]]
    N, n = 128, 10
    orders = []
    for k in ("eps_1", "eps_2", "eps_3"):
        top = np.array(rec[k], dtype=np.int32)
        rest = np.setdiff1d(np.arange(N, dtype=np.int32), top)
        orders.append(_t(np.concatenate([top, rest])[None, :]))
    u_min = torch.stack([snaps.topn_overlap(orders[0], o, n) for o in orders])
    u_max = torch.stack([snaps.topn_overlap(orders[2], o, n) for o in orders])
    j = snaps.select_parameter(u_min.contiguous(), u_max.contiguous(), n)
    torch.cuda.synchronize()
    assert np.allclose(u_min[:, 0].cpu().numpy(), rec["U_min"]) and np.allclose(u_max[:, 0].cpu().numpy(), rec["U_max"])
    assert int(j[0]) == 1


def test_k_grid_pipeline_matches_oracle(snaps):
    """k_max join once, then every k_j of a grid from its prefix, ranking, Eq. 2 and
    Eq. 3 -- device against the oracle functions on the same lists."""
    import torch
    N, k_max, n = 3000, 32, 30                      # n = 1% of N
    X = workloads.make_table(N, 17, outlier_frac=0.01)
    masks = workloads.all_masks(15)[::2111]
    join = snaps.knn_selfjoin(_t(X), masks, k_max, scores=False)
    torch.cuda.synchronize()
    idx, dist = join["idx"].cpu().numpy(), join["dist"].cpu().numpy()
    grid = [2, 3, 5, 8, 12, 20, 32]
    for metric, key in (("knn_indegree", "indeg"), ("knn_mean", "mean")):
        orders = []
        for kj in grid:
            sc = snaps.knn_scores_at_k(join["idx"], join["dist"], kj)
            torch.cuda.synchronize()
            for m in range(len(masks)):
                kth, mean, indeg = oracle_ranking.knn_scores_at_k(idx[m], dist[m], kj, N)
                assert (sc["indeg"][m].cpu().numpy() == indeg).all()
                assert np.allclose(sc["kth"][m].cpu().numpy(), kth, rtol=1e-6)
                assert np.allclose(sc["mean"][m].cpu().numpy(), mean, rtol=1e-5)
            orders.append(snaps.rank_scores(metric, sc[key].contiguous(), ranks=False)["order"])
        u_min = torch.stack([snaps.topn_overlap(orders[0], o, n) for o in orders]).contiguous()
        u_max = torch.stack([snaps.topn_overlap(orders[-1], o, n) for o in orders]).contiguous()
        sel = snaps.select_parameter(u_min, u_max, n)
        torch.cuda.synchronize()
        for m in range(len(masks)):
            tops = [o[m, :n].cpu().numpy() for o in orders]
            o_min, o_max = oracle_ranking.similarity_curves(tops, n)
            assert np.allclose(u_min[:, m].cpu().numpy(), o_min) and np.allclose(u_max[:, m].cpu().numpy(), o_max)
            assert int(sel[m]) == oracle_ranking.select_parameter(o_min, o_max, n)
        assert float(u_min[0].min()) == 1.0 and float(u_max[-1].min()) == 1.0     # a set against itself


def test_radius_grid_single_scan_matches_oracle_per_radius(snaps):
    """PAPER.md:235-239 (Fig. 3): one join at eps_max gives the result for every eps_j of the grid.
    The oracle is the definition evaluated once per radius (no shared work)."""
    import sys
    import torch
    sys.path.insert(0, HERE)
    from parity import check_range
    import oracle as oracle_mod
    X = workloads.make_table(1500, 29, outlier_frac=0.01)
    masks = np.array([0b11, 0x7FFF, (1 << 7) | (1 << 2) | 1, 0b111100, (1 << 14) | (1 << 9)], dtype=np.uint16)
    scale = np.array([1.0, 6.0, 2.0, 3.0, 1.5], dtype=np.float32)
    G = 7
    grid = (np.linspace(0.015, 0.12, G, dtype=np.float32)[None, :] * scale[:, None]).astype(np.float32)
    out = snaps.range_selfjoin_grid(_t(X), masks, grid)
    torch.cuda.synchronize()
    cnt = out["count"].cpu().numpy()
    for g in range(G):
        check_range(cnt[:, g], out["sumdist"][:, g].cpu().numpy(), out["mean"][:, g].cpu().numpy(),
                    oracle_mod, X, masks, grid[:, g])
    assert (np.diff(cnt, axis=1) >= 0).all()                      # nested result sets
    # the single-radius entry point gives the same counts
    one = snaps.range_selfjoin(_t(X), masks, grid[:, 3])
    torch.cuda.synchronize()
    assert (one["count"].cpu().numpy() == cnt[:, 3]).all()
    with pytest.raises(snaps.SnapsError):
        snaps.range_selfjoin_grid(_t(X), masks, grid[:, ::-1].copy())   # not ascending


@pytest.mark.parametrize("engine", ["lattice", "grid"])
def test_radius_grid_irregular_radii(snaps, engine):
    """The kernels guess a neighbour's radius bin as if the radii were evenly spaced and settle the guess against
    the exact thresholds: grids that are anything but evenly spaced (geometric, clustered at either end, radii a few
    ulps apart, G = 1, 2 and the maximum 32) must give, radius by radius, exactly the counts of the single-radius join
    and its sums within the fp32 summation-order tolerance."""
    import torch
    rng = np.random.default_rng(77)
    X = workloads.make_table(1300, 31, outlier_frac=0.02)
    masks = np.array([0b11, 0x7FFF, (1 << 11) | (1 << 4) | 0b10, 0b1111100, (1 << 13) | (1 << 6), 0b101], dtype=np.uint16)
    scale = np.array([1.0, 6.0, 2.0, 3.0, 1.5, 1.2], dtype=np.float32)
    Xd = _t(X)
    grids = {
        "geometric": np.geomspace(0.004, 0.16, 12),
        "clustered_low": np.concatenate([np.linspace(0.01, 0.012, 9), [0.05, 0.15]]),
        "clustered_high": np.concatenate([[0.005, 0.03], np.linspace(0.140, 0.141, 10)]),
        "adjacent_floats": np.array([0.02, 0.0200001, 0.0200002, 0.07, 0.0700001, 0.13]),
        "one": np.array([0.06]),
        "two": np.array([0.001, 0.2]),
        "thirty_two": np.sort(rng.uniform(0.002, 0.18, 32)),
    }
    for name, base in grids.items():
        grid = (base[None, :].astype(np.float32) * scale[:, None]).astype(np.float32)
        out = snaps.range_selfjoin_grid(Xd, masks, grid, engine=engine)
        torch.cuda.synchronize()
        cnt, sm = out["count"].cpu().numpy(), out["sumdist"].cpu().numpy()
        assert (np.diff(cnt, axis=1) >= 0).all(), name
        for g in sorted({0, grid.shape[1] // 2, grid.shape[1] - 1}):
            one = snaps.range_selfjoin(Xd, masks, grid[:, g], engine=engine)
            torch.cuda.synchronize()
            assert np.array_equal(one["count"].cpu().numpy(), cnt[:, g]), (name, g)
            ref = one["sumdist"].cpu().numpy()
            assert np.allclose(sm[:, g], ref, rtol=3e-5, atol=1e-6), (name, g)


def test_select_k_pipeline_matches_oracle(snaps):
    """snaps_knn_select_k (one call: k grid -> scores -> ranks -> Eq. 2 -> Eq. 3) against the oracle
    procedure, mask by mask, on the SAME k_max lists: the oracle's own join, cast to the fp32 lists the
    device call takes.  Index work: U curves and selected grid points are compared exactly; the ranks by
    mean distance are decided on the fp32 mean on both sides (reading A21)."""
    import torch
    import oracle as oracle_mod
    N, k_max, n = 2500, 32, 25
    X = workloads.make_table(N, 31, outlier_frac=0.01)
    masks = workloads.all_masks(15)[::1409]
    oi, od = oracle_mod.knn_selfjoin(X, masks, k_max)
    idx, dist = oi.astype(np.int32), od.astype(np.float32)
    grid = [2, 3, 4, 6, 8, 11, 16, 23, 32]
    out = snaps.knn_select_k(_t(idx), _t(dist), grid, n)
    torch.cuda.synchronize()
    u = out["u"].cpu().numpy()
    for m in range(len(masks)):
        ref = oracle_ranking.select_k(idx[m], dist[m], grid, n, N)
        ji, umin_i, umax_i = ref["knn_indegree"]
        assert np.array_equal(u[0][:, m], umin_i.astype(np.float32)) and np.array_equal(u[1][:, m], umax_i.astype(np.float32))
        assert int(out["j_indeg"][m]) == ji
        jm, umin_m, umax_m = ref["knn_mean"]
        assert np.array_equal(u[2][:, m], umin_m.astype(np.float32)) and np.array_equal(u[3][:, m], umax_m.astype(np.float32))
        assert int(out["j_mean"][m]) == jm
    assert (u[0][0] == 1.0).all() and (u[1][-1] == 1.0).all() and (u[2][0] == 1.0).all() and (u[3][-1] == 1.0).all()
    # the same call on the device's own lists runs end to end (join -> selection without leaving the GPU)
    join = snaps.knn_selfjoin(_t(X), masks, k_max, scores=False)
    out2 = snaps.knn_select_k(join["idx"], join["dist"], grid, n)
    torch.cuda.synchronize()
    assert (out2["j_indeg"].cpu().numpy() == out["j_indeg"].cpu().numpy()).mean() > 0.9
    with pytest.raises(snaps.SnapsError):
        snaps.knn_select_k(join["idx"], join["dist"], [4, 2, 8], n)


def test_sampled_distance_histogram_and_eps_search(snaps):
    """NEXT-2: device histogram of sampled pair distances against the oracle's,
    bin by bin (pairs within 1e-6 relative of a bin edge may fall on either side: fp32 vs fp64),
    and the radius for a target selectivity from its cumulative form."""
    import torch
    from oracle.calibrate import sampled_histogram, eps_from_histogram
    N = 4000
    X = workloads.make_table(N, 37, outlier_frac=0.01)
    masks = np.array([0b11, 0x7FFF, (1 << 9) | (1 << 3) | 1, 0b1111000], dtype=np.uint16)
    rng = np.random.default_rng(5)
    q = np.sort(rng.choice(N, 300, replace=False)).astype(np.int32)
    c = np.sort(rng.choice(N, 1500, replace=False)).astype(np.int32)
    rmax = np.array([0.05, 0.6, 0.2, 0.3], dtype=np.float32)
    n_bins = 256
    hist = snaps.sample_distance_histogram(_t(X), masks, q, c, rmax, n_bins)
    torch.cuda.synchronize()
    g = hist.cpu().numpy()
    ref, dists = sampled_histogram(X, masks, q, c, rmax, n_bins)
    for mi in range(len(masks)):
        edges = np.arange(1, n_bins + 1) * (float(rmax[mi]) / n_bins)
        d = dists[mi]
        # cumulative counts may differ by the pairs inside the band around each edge
        lo = np.array([(d < e * (1 - 1e-6)).sum() for e in edges])
        hi = np.array([(d < e * (1 + 1e-6)).sum() for e in edges])
        cum = np.cumsum(g[mi])
        assert (lo <= cum).all() and (cum <= hi).all()
        assert np.abs(g[mi] - ref[mi]).sum() <= 2 * (hi - lo).sum()
    pairs = int(sum(len(c) - int(qq in set(c.tolist())) for qq in q))
    e_dev = snaps.eps_from_histogram(g, rmax, N, pairs, 20.0)
    e_ref = eps_from_histogram(ref, rmax, N, pairs, 20.0)
    assert np.abs(e_dev - e_ref).max() <= (rmax / n_bins).max() * 1.001        # at most one bin apart
    # the radius does what it is for: the eps-join at it finds about the target number of neighbours
    cnt = snaps.range_selfjoin(_t(X), masks, e_dev)["count"].float().mean(dim=1).cpu().numpy()
    assert (cnt > 10).all() and (cnt < 40).all()


def test_eps_search_matches_oracle(snaps):
    """snaps_eps_search (PAPER.md:229-237 in one device call: eps_mean, histogram over [0, eps_mean), radii
    for two target selectivities) against oracle.calibrate.eps_search, step by step."""
    import torch
    from oracle.calibrate import eps_search
    N = 3000
    X = workloads.make_table(N, 41, outlier_frac=0.01)
    masks = np.array([0b11, 0x7FFF, (1 << 9) | (1 << 3) | 1, 0b1111000, (1 << 13) | (1 << 12)], dtype=np.uint16)
    rng = np.random.default_rng(9)
    q = np.sort(rng.choice(N, 200, replace=False)).astype(np.int32)
    c = np.sort(rng.choice(N, 1200, replace=False)).astype(np.int32)
    n_bins, targets = 512, [3.0, 450.0]          # s_min ~ 0.001 |D|, s_max ~ 0.15 |D|
    out = snaps.eps_search(_t(X), masks, q, c, targets, n_bins, hist=True)
    torch.cuda.synchronize()
    rmax, eps, hist, dists = eps_search(X, masks, q, c, n_bins, targets)
    g_mean = out["eps_mean"].cpu().numpy()
    assert np.abs(g_mean - rmax).max() <= 2e-6 * rmax.max()                   # fp32 value of an fp64-accumulated mean
    g_hist = out["hist"].cpu().numpy()
    for mi in range(len(masks)):
        edges = np.arange(1, n_bins + 1) * (float(rmax[mi]) / n_bins)
        lo = np.array([(dists[mi] < e * (1 - 2e-6)).sum() for e in edges])
        hi = np.array([(dists[mi] < e * (1 + 2e-6)).sum() for e in edges])
        cum = np.cumsum(g_hist[mi])
        assert (lo <= cum).all() and (cum <= hi).all()
    g_eps = out["eps"].cpu().numpy()
    assert np.abs(g_eps - eps).max() <= (rmax / n_bins).max() * 1.001          # at most one bin apart
    assert (np.abs(g_eps - eps) <= 1e-6 * eps).mean() >= 0.8                   # and mostly the same edge
    assert (g_eps[:, 0] < g_eps[:, 1]).all() and (g_eps[:, 1] <= g_mean * 1.000001).all()
    # the radii do what they are for
    for t, col in zip(targets, (0, 1)):
        cnt = snaps.range_selfjoin(_t(X), masks, g_eps[:, col], sums=False)["count"].float().mean(dim=1).cpu().numpy()
        assert (cnt > 0.5 * t).all() and (cnt < 2.0 * t).all(), (t, cnt)


@pytest.mark.parametrize("engine", ["lattice", "grid"])
def test_select_eps_pipeline_matches_oracle(snaps, engine):
    """snaps_range_select_eps (one call: eps_min / eps_max search -> eps grid -> one join at eps_max -> ranks
    -> Eq. 2 -> Eq. 3) against the oracle procedure written out step by step (calibrate.eps_search,
    ranking.eps_grid, one range join per radius, ranking.select_eps), mask by mask.  Index work is compared
    exactly wherever no pair sits within 1e-6 of a grid radius (reading A2) and, for the mean-distance
    metric, no object sits within 1e-5 relative of the top-n boundary (near-tie rule: the device mean is an
    fp32 sum in scan order)."""
    import torch
    import oracle as oracle_mod
    from oracle.calibrate import eps_search
    N, G, n = 1800, 8, 18
    X = workloads.make_table(N, 43, outlier_frac=0.01)
    masks = np.array([0b11, 0x7FFF, (1 << 9) | (1 << 3) | 1, 0b1111000, (1 << 13) | (1 << 12), 0b111111], dtype=np.uint16)
    rng = np.random.default_rng(11)
    q = np.sort(rng.choice(N, 300, replace=False)).astype(np.int32)
    c = np.arange(N, dtype=np.int32)
    s_min, s_max, n_bins = 0.002 * N, 0.15 * N, 1024
    out = snaps.range_select_eps(_t(X), masks, q, c, s_min, s_max, G, n, n_bins, engine=engine)
    torch.cuda.synchronize()
    _, eps, _, _ = eps_search(X, masks, q, c, n_bins, [s_min, s_max])
    u = out["u"].cpu().numpy()
    g_grid = out["eps_grid"].cpu().numpy()
    exact_masks = 0
    for m in range(len(masks)):
        grid = oracle_ranking.eps_grid(eps[m, 0], eps[m, 1], G)
        assert np.abs(g_grid[m] - grid).max() <= 2e-6 * grid.max()
        one = np.array([masks[m]] * G, dtype=np.uint16)
        cnt, _, mean = oracle_mod.range_selfjoin(X, one, grid.astype(np.float64))
        # the device's radii may sit an fp32 rounding or two from the oracle's (asserted above): widen the band of A2
        lo, _, _ = oracle_mod.range_selfjoin(X, one, grid.astype(np.float64) * (1 - 4e-6))
        hi, _, _ = oracle_mod.range_selfjoin(X, one, grid.astype(np.float64) * (1 + 4e-6))
        ref = oracle_ranking.select_eps(cnt, mean, n)
        jc, umin_c, umax_c = ref["dssj_count"]
        # exactness is asked for where the band cannot move a top-n set: the n objects with the fewest neighbours
        # are the same whether the pairs inside the band are counted or not
        tops = lambda c: [set(oracle_ranking.topn_ids("dssj_count", c[g], n).tolist()) for g in range(G)]
        if tops(lo) == tops(cnt) == tops(hi):
            exact_masks += 1
            assert np.array_equal(u[0][:, m], umin_c.astype(np.float32)) and np.array_equal(u[1][:, m], umax_c.astype(np.float32))
            assert int(out["j_count"][m]) == jc
            # mean-distance metric: exact unless an object sits on the top-n boundary of some radius or a band
            # pair touches one of the top-n objects
            near = 0
            for g in range(G):
                key = np.where(cnt[g] == 0, np.inf, mean[g])           # most outlying first = descending
                srt = np.sort(key)[::-1]
                b = srt[n - 1]
                near += int((np.abs(key - b) <= 1e-5 * max(b, 1e-30)).sum() - 1) if np.isfinite(b) else 0
                top = oracle_ranking.topn_ids("dssj_mean", mean[g], n + 2, counts=cnt[g])
                near += int((lo[g][top] != hi[g][top]).sum())
            jm, umin_m, umax_m = ref["dssj_mean"]
            if near == 0:
                assert np.array_equal(u[2][:, m], umin_m.astype(np.float32)) and np.array_equal(u[3][:, m], umax_m.astype(np.float32))
                assert int(out["j_mean"][m]) == jm
            else:
                assert np.abs(u[2][:, m] - umin_m).max() <= near / n and np.abs(u[3][:, m] - umax_m).max() <= near / n
    assert exact_masks >= len(masks) - 1
    assert (u[0][0] == 1.0).all() and (u[1][-1] == 1.0).all() and (u[2][0] == 1.0).all() and (u[3][-1] == 1.0).all()


def test_range_from_knn_matches_oracle_and_the_range_join(snaps):
    """snaps_range_from_knn (PAPER.md:537 kNN -> DSSJ reuse): index work against the oracle function on the same
    lists (exact), and against the device's own eps-join wherever the list is complete."""
    import torch
    import oracle as oracle_mod
    N, k = 3000, 24
    X = workloads.make_table(N, 47, outlier_frac=0.01)
    masks = np.array([0b11, 0x7FFF, (1 << 9) | (1 << 3) | 1, 0b1111000], dtype=np.uint16)
    _, od = oracle_mod.knn_selfjoin(X, masks, k)
    dist = od.astype(np.float32)
    eps = np.array([np.median(dist[m, :, 9]) * 1.0003 for m in range(len(masks))], dtype=np.float32)
    out = snaps.range_from_knn(_t(dist), eps)
    torch.cuda.synchronize()
    for m in range(len(masks)):
        cnt, s, mean, complete = oracle_ranking.range_from_knn(dist[m], eps[m])
        assert (out["count"][m].cpu().numpy() == cnt).all() and (out["complete"][m].cpu().numpy() == complete).all()
        assert np.allclose(out["sumdist"][m].cpu().numpy(), s, rtol=1e-5) and np.allclose(out["mean"][m].cpu().numpy(), mean, rtol=1e-5)
    # on the device's own lists: complete objects need no range join
    Xd = _t(X)
    join = snaps.knn_selfjoin(Xd, masks, k, scores=False)
    reuse = snaps.range_from_knn(join["dist"], eps)
    rj = snaps.range_selfjoin(Xd, masks, eps)
    torch.cuda.synchronize()
    c = reuse["complete"].bool()
    assert 0.2 < c.float().mean().item() < 0.9
    agree = (reuse["count"][c] == rj["count"][c]).float().mean().item()
    assert agree > 0.999                                            # all but pairs inside the 1e-6 band of A2
    assert bool((reuse["count"][~c] == k).all()) and bool((rj["count"][~c] >= k).all())
