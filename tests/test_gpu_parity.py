"""GPU parity: libsnaps (through the C ABI binding) against the fp64 oracle, element by element."""
import numpy as np
import pytest

import workloads
from parity import check_knn, check_knn_scores, check_range

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def snaps():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2405_20176_b200 as s
    s.lib()
    return s


def _dev(X):
    import torch
    return torch.from_numpy(np.ascontiguousarray(X)).cuda()


def _knn_case(snaps, oracle_mod, X, masks, k, engine="auto"):
    import torch
    out = snaps.knn_selfjoin(_dev(X), masks, k, engine=engine)
    torch.cuda.synchronize()
    g = {n: out[n].cpu().numpy() for n in ("idx", "dist", "kth", "mean", "indeg")}
    N = len(X)
    kk = min(k + 1, N - 1)
    oi, od = oracle_mod.knn_selfjoin(X, masks, kk)
    if kk == k:                                   # no (k+1)-th neighbour exists: nothing is ambiguous
        oi = np.concatenate([oi, np.full(oi.shape[:2] + (1,), -1, oi.dtype)], axis=2)
        od = np.concatenate([od, np.full(od.shape[:2] + (1,), np.inf)], axis=2)
    unamb = check_knn(g["idx"], g["dist"], oi, od)
    kth, mean, indeg = oracle_mod.knn_scores(N, oi[:, :, :k], od[:, :, :k])
    check_knn_scores(g, g["idx"], kth, mean, indeg, unamb, N)
    return g, unamb


def test_config1_tiny_full(snaps, oracle_mod):
    cfg = workloads.get_config("c1_tiny")
    g, unamb = _knn_case(snaps, oracle_mod, cfg.table(), cfg.masks(), cfg.k)
    assert unamb.mean() > 0.99


@pytest.mark.parametrize("n,nf,k,seed", [
    (2, 2, 1, 0), (3, 3, 2, 1), (33, 4, 5, 2), (127, 7, 10, 3), (128, 15, 10, 4), (129, 15, 16, 5),
    (300, 15, 32, 6), (1000, 12, 3, 7), (1537, 15, 10, 8),
])
def test_knn_ragged_sizes(snaps, oracle_mod, n, nf, k, seed):
    X = workloads.make_table(n, seed, cols=list(range(nf)), outlier_frac=0.02)
    allm = workloads.all_masks(nf, 1)
    rng = np.random.default_rng(seed)
    masks = rng.choice(allm, min(len(allm), 40), replace=False)
    _knn_case(snaps, oracle_mod, X, masks, k)


def test_knn_all_masks_9_features(snaps, oracle_mod):
    # several batches (H over 3 high features), every lattice slot used
    X = workloads.make_table(700, 11, cols=list(range(9)))
    _knn_case(snaps, oracle_mod, X, workloads.all_masks(9, 1), 10)


def test_knn_hypercube_ties(snaps, oracle_mod):
    # massive exact ties (closed form B): distances must match, ids only need to be valid
    X = workloads.hypercube_table(9)
    masks = workloads.all_masks(9, 1)[::7]
    _knn_case(snaps, oracle_mod, X, masks, 10)


def test_knn_duplicate_block(snaps, oracle_mod):
    # readings A4/A7: other objects at distance 0 are neighbours; ties go to the smaller id
    X = workloads.duplicate_block_table(900, 3, frac=0.3)
    masks = np.array([(1 << 13) | (1 << 14), (1 << 13) | 1, 0x7FFF, 1 << 14], dtype=np.uint16)
    g, _ = _knn_case(snaps, oracle_mod, X, masks, 10)
    oi, od = oracle_mod.knn_selfjoin(X, masks, 10)
    # a distance-0 block: exact same ids as the oracle (tie-break by id is deterministic)
    zero = od[0, :, -1] == 0
    assert zero.sum() > 100 and (g["idx"][0][zero] == oi[0][zero]).all()


def test_knn_scores_only_and_lists_only(snaps, oracle_mod):
    import torch
    X = workloads.make_table(500, 21, cols=list(range(8)))
    masks = workloads.all_masks(8)[::5]
    Xd = _dev(X)
    full = snaps.knn_selfjoin(Xd, masks, 6)
    so = snaps.knn_selfjoin(Xd, masks, 6, lists=False)
    lo = snaps.knn_selfjoin(Xd, masks, 6, scores=False)
    torch.cuda.synchronize()
    assert "idx" not in so and "kth" not in lo
    for n in ("kth", "mean", "indeg"):
        assert torch.equal(full[n], so[n])
    for n in ("idx", "dist"):
        assert torch.equal(full[n], lo[n])
    # determinism: a second run is bit-identical
    again = snaps.knn_selfjoin(Xd, masks, 6)
    torch.cuda.synchronize()
    for n in ("idx", "dist", "kth", "mean", "indeg"):
        assert torch.equal(full[n], again[n])


def test_outlier_scores_entry_point(snaps, oracle_mod):
    import torch
    X = workloads.make_table(400, 5, cols=list(range(6)))
    masks = workloads.all_masks(6)
    Xd = _dev(X)
    j = snaps.knn_selfjoin(Xd, masks, 7)
    r = snaps.range_selfjoin(Xd, masks, np.full(len(masks), 0.08, np.float32))
    s = snaps.outlier_scores(400, len(masks), 7, knn_idx=j["idx"], knn_dist=j["dist"],
                             eps_count=r["count"], eps_sumdist=r["sumdist"])
    torch.cuda.synchronize()
    assert torch.equal(s["kth"], j["kth"]) and torch.equal(s["indeg"], j["indeg"])
    assert torch.allclose(s["mean"], j["mean"], rtol=1e-6, atol=0)
    assert torch.equal(s["eps_mean"], r["mean"])
    oi, od = oracle_mod.knn_selfjoin(X, masks, 7)
    kth, mean, indeg = oracle_mod.knn_scores(400, oi, od)
    np.testing.assert_allclose(s["kth"].cpu().numpy(), kth, rtol=1e-4, atol=1e-7)


@pytest.mark.parametrize("n,nf,seed,sums", [(2, 2, 0, True), (130, 5, 1, True), (1000, 15, 2, True),
                                            (1537, 15, 3, False), (640, 9, 4, True)])
def test_range_join(snaps, oracle_mod, n, nf, seed, sums):
    import torch
    X = workloads.make_table(n, seed, cols=list(range(nf)), outlier_frac=0.02)
    allm = workloads.all_masks(nf, 1)
    rng = np.random.default_rng(seed)
    masks = rng.choice(allm, min(len(allm), 48), replace=False)
    kq = min(10, n - 1)
    _, od = oracle_mod.knn_selfjoin(X, masks, kq)
    # 1.003x: keep eps off the realised pair distance the median sits on (tiny n would put that
    # pair inside the 1e-6 band of reading A2)
    eps = np.array([max(1.003 * np.median(od[m, :, -1]), 1e-3) for m in range(len(masks))], dtype=np.float32)
    out = snaps.range_selfjoin(_dev(X), masks, eps, sums=sums)
    torch.cuda.synchronize()
    cnt = out["count"].cpu().numpy()
    lo, hi = check_range(cnt, out["sumdist"].cpu().numpy() if sums else None,
                         out["mean"].cpu().numpy() if sums else None, oracle_mod, X, masks, eps)
    assert (lo == hi).mean() > 0.99
    # symmetric join: total count is even wherever no pair sits in the band
    for m in range(len(masks)):
        if (lo[m] == hi[m]).all():
            assert cnt[m].sum() % 2 == 0


def test_range_hypercube_closed_form(snaps, oracle_mod):
    import torch
    from scipy.special import comb
    X = workloads.hypercube_table(9)
    masks = workloads.all_masks(9, 1)[::5]
    eps = np.full(len(masks), 1.5, np.float32)
    out = snaps.range_selfjoin(_dev(X), masks, eps)
    torch.cuda.synchronize()
    cnt = out["count"].cpu().numpy()
    for mi, m in enumerate(masks):
        d = bin(int(m)).count("1")
        mult = 1 << (9 - d)
        exp = sum(comb(d, r, exact=True) * mult for r in range(d + 1) if r ** 0.5 <= 1.5) - 1
        assert (cnt[mi] == exp).all()


def test_streamed_matches_resident(snaps, oracle_mod):
    import torch
    X = workloads.make_table(1200, 31, cols=list(range(10)))
    masks = workloads.all_masks(10)[::9]
    Xd = _dev(X)
    ref = snaps.knn_selfjoin(Xd, masks, 10)
    st = snaps.knn_selfjoin_streamed(Xd, masks, 10, masks_per_batch=17)
    torch.cuda.synchronize()
    for n in ("idx", "dist", "kth", "mean", "indeg"):
        assert st[n].is_pinned()
        assert torch.equal(st[n], ref[n].cpu()), n
    host = snaps.knn_selfjoin_host(X, masks, 10, masks_per_batch=50, lists=True)
    torch.cuda.synchronize()
    assert torch.equal(host["kth"], ref["kth"].cpu()) and torch.equal(host["idx"], ref["idx"].cpu())


def test_strided_input_and_stream(snaps, oracle_mod):
    import torch
    X = workloads.make_table(333, 41, cols=list(range(5)))
    wide = torch.zeros((333, 9), dtype=torch.float32, device="cuda")
    wide[:, :5] = _dev(X)
    view = wide[:, :5]                      # row stride 9 floats
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        out = snaps.knn_selfjoin(view, [0b10101, 0b11111], 4, stream=s)
    s.synchronize()
    oi, od = oracle_mod.knn_selfjoin(X, [0b10101, 0b11111], 5)
    check_knn(out["idx"].cpu().numpy(), out["dist"].cpu().numpy(), oi, od)


def test_argument_errors(snaps):
    import torch
    X = torch.rand((10, 4), device="cuda")
    with pytest.raises(snaps.SnapsError) as e:
        snaps.knn_selfjoin(X, [0b1111], 10)              # k > N-1 (reading A9)
    assert e.value.status == 1
    with pytest.raises(snaps.SnapsError):
        snaps.knn_selfjoin(X, [0], 3)                    # zero mask
    with pytest.raises(snaps.SnapsError):
        snaps.knn_selfjoin(X, [0b10000], 3)              # bit >= n_feat
    with pytest.raises(snaps.SnapsError):
        snaps.knn_selfjoin(X, [0b11], 4097)              # k > SNAPS_MAX_K
    with pytest.raises(snaps.SnapsError):
        snaps.knn_selfjoin(torch.rand((600, 4), device="cuda"), [0b11], 300, lists=False)   # k > 256 builds the lists in place
    with pytest.raises(snaps.SnapsError):
        snaps.range_selfjoin(X, [0b11], [float("nan")])
    with pytest.raises(snaps.SnapsError):
        snaps.range_selfjoin(X, [0b11], [0.0])
    with pytest.raises(snaps.SnapsError) as e:
        snaps.knn_selfjoin(X, [0b11], 3, workspace=torch.empty(256, dtype=torch.uint8, device="cuda"))
    assert e.value.status == 3
    with pytest.raises(snaps.SnapsError):
        snaps.knn_selfjoin(X, [0b11], 3, lists=False, scores=False)


# ---------------------------------------------------------------- full-size configs, sampled outputs
def _sampled_knn_check(snaps, oracle_mod, cfg, out, X, masks, n_masks_s, n_queries_s, seed):
    """Compare kth/mean of a scores-only full-size run with the oracle on sampled (mask, query)
    rows (a kNN row does not depend on other queries, so per-row sampling is exact)."""
    rng = np.random.default_rng(seed)
    pc = workloads.popcount(masks)
    ms = np.sort(np.concatenate([rng.choice(np.flatnonzero(pc == d), min(2, int((pc == d).sum())), replace=False)
                                 for d in np.unique(pc)]))[:n_masks_s]
    qs = np.sort(rng.choice(len(X), n_queries_s, replace=False))
    oi, od = oracle_mod.knn_selfjoin(X, masks[ms], cfg.k, queries=qs)
    kth = out["kth"][ms][:, qs].cpu().numpy().astype(np.float64)
    mean = out["mean"][ms][:, qs].cpu().numpy().astype(np.float64)
    assert (np.abs(kth - od[:, :, -1]) <= 1e-4 * od[:, :, -1] + 1e-7).all()
    assert (np.abs(mean - od.mean(axis=2)) <= 1e-4 * od.mean(axis=2) + 1e-7).all()
    return ms, qs


def test_config2_full_size_sampled(snaps, oracle_mod):
    """BASELINE.json configs[1] exactly as bench.py launches it (N=31,693, 32,752 masks, k=10,
    scores only).  SURVEY 8(c) oracle tiers: ALL masks x 16 sampled queries (every one of the 512 batches
    and every lattice slot), whole-output invariants, the in-degree of two complete masks against a full
    oracle join, and ids + distances of eight whole batches (512 masks) x 256 sampled queries through the
    streamed call."""
    import torch
    cfg = workloads.get_config("c2_snapshot1_knn")
    X, masks = cfg.table(), cfg.masks()
    N, k = len(X), cfg.k
    Xd = _dev(X)
    out = snaps.knn_selfjoin(Xd, masks, k, lists=False)
    torch.cuda.synchronize()
    rng = np.random.default_rng(5)
    qs = np.sort(rng.choice(N, 16, replace=False))
    oi, od = oracle_mod.knn_selfjoin(X, masks, k, queries=qs)          # all 32,752 masks
    kth = out["kth"][:, qs].cpu().numpy().astype(np.float64)
    mean = out["mean"][:, qs].cpu().numpy().astype(np.float64)
    assert (np.abs(kth - od[:, :, -1]) <= 1e-4 * od[:, :, -1] + 1e-7).all()
    assert (np.abs(mean - od.mean(axis=2)) <= 1e-4 * od.mean(axis=2) + 1e-7).all()
    # invariants over the whole output (mean <= kth; monotone along lattice edges)
    assert bool((out["indeg"].sum(dim=1) == N * k).all())
    assert bool((out["mean"] <= out["kth"] * (1 + 1e-6)).all()) and bool((out["kth"] > 0).all())
    pos = {int(m): i for i, m in enumerate(masks)}
    for m in rng.choice(masks, 40, replace=False):
        for f in range(15):
            sup = int(m) | (1 << f)
            if sup != int(m):
                a, b = out["kth"][pos[int(m)]], out["kth"][pos[sup]]
                assert bool((a <= b * (1 + 1e-5) + 1e-7).all())      # D_(k)(S) <= D_(k)(S u {f})
    # in-degree: two complete masks, full oracle join
    for mi in (int(rng.integers(len(masks))), len(masks) - 1):
        oi1, od1 = oracle_mod.knn_selfjoin(X, masks[mi:mi + 1], k + 1)
        unamb = (od1[0, :, k] - od1[0, :, k - 1]) > 1e-5 * od1[0, :, k]
        hist = np.bincount(oi1[0, :, :k].ravel(), minlength=N)
        got = out["indeg"][mi].cpu().numpy()
        if unamb.all():
            assert (got == hist).all()
        else:   # only ambiguous queries' k-th neighbours may differ
            assert np.abs(got - hist).sum() <= 2 * (~unamb).sum()
    del out
    # ids + distances: eight whole batches (all 64 lattice slots of eight sets H), streamed in groups of 100 masks
    hs = rng.choice(np.unique(masks.astype(np.int64) >> 6), 8, replace=False)
    sel = np.flatnonzero(np.isin(masks.astype(np.int64) >> 6, hs))
    assert 8 * 57 <= len(sel) <= 8 * 64
    st = snaps.knn_selfjoin_streamed(Xd, masks[sel], k, masks_per_batch=100, lists=True)
    torch.cuda.synchronize()
    qs2 = np.sort(rng.choice(N, 256, replace=False))
    oi2, od2 = oracle_mod.knn_selfjoin(X, masks[sel], k + 1, queries=qs2)
    check_knn(st["idx"][:, qs2].numpy(), st["dist"][:, qs2].numpy(), oi2, od2, queries=qs2)


def test_config3_full_size_sampled(snaps, oracle_mod):
    """BASELINE.json configs[2] as bench.py launches it: DSSJ over all 32,752 masks at N=31,693 with the
    stored per-dimension eps_d (~50 neighbours; workloads/config_eps.json); ALL masks x 16 sampled queries
    against the oracle, plus invariants."""
    import torch
    cfg = workloads.get_config("c3_snapshot1_dssj")
    X, masks = cfg.table(), cfg.masks()
    N = len(X)
    eps = workloads.config_eps(cfg.name, masks)
    out = snaps.range_selfjoin(_dev(X), masks, eps)
    torch.cuda.synchronize()
    rng = np.random.default_rng(7)
    qs = np.sort(rng.choice(N, 16, replace=False))
    check_range(out["count"][:, qs].cpu().numpy(), out["sumdist"][:, qs].cpu().numpy(), out["mean"][:, qs].cpu().numpy(),
                oracle_mod, X, masks, eps, queries=qs)
    mean_cnt = out["count"].float().mean().item()
    assert 10 < mean_cnt < 250, mean_cnt                     # calibrated for ~50 (sample noise allowed)
    # no self-pairs, counts bounded by N-1; the mean is 0 exactly where the count is 0 (A6)
    assert int(out["count"].max().item()) <= N - 1
    assert bool((out["mean"][out["count"] == 0] == 0).all())


def test_streamed_large_table_reduced_configs_4_5(snaps, oracle_mod):
    """Configs 4-5 in shape (pair masks + full set; 256 sampled masks, k=16) on a reduced N, through
    the pinned-host streaming call; sampled rows against the oracle."""
    import torch
    for name, n, k, masks in (("c4", 60_000, 10, workloads.pair_masks_plus_full(15)),
                              ("c5", 40_000, 16, workloads.sample_masks(256, 4)[::4])):
        X = workloads.make_table(n, 3, outlier_frac=0.001)
        st = snaps.knn_selfjoin_streamed(_dev(X), masks, k, masks_per_batch=16, lists=True)
        torch.cuda.synchronize()
        rng = np.random.default_rng(8)
        qs = np.sort(rng.choice(n, 24, replace=False))
        sel = np.arange(len(masks))[:: max(1, len(masks) // 12)]
        oi, od = oracle_mod.knn_selfjoin(X, masks[sel], k + 1, queries=qs)
        check_knn(st["idx"][sel][:, qs].numpy(), st["dist"][sel][:, qs].numpy(), oi, od, queries=qs)
        assert bool((st["indeg"].sum(dim=1) == n * k).all())


# ---------------------------------------------------------------- grid engine (large N, arbitrary masks, k <= 256)
# The library takes the grid engine at N >= 2^18 or k > 32; engine="grid" forces it so that the path
# is checked element by element at sizes the oracle finishes in seconds.
@pytest.mark.parametrize("n,nf,k,seed", [(2, 2, 1, 0), (3, 3, 2, 1), (33, 4, 5, 2), (129, 15, 16, 5), (1537, 15, 10, 8),
                                         (3000, 12, 3, 7), (700, 9, 10, 11), (5000, 15, 16, 12)])
def test_grid_engine_random_tables(snaps, oracle_mod, n, nf, k, seed):
    X = workloads.make_table(n, seed, cols=list(range(nf)), outlier_frac=0.02)
    allm = workloads.all_masks(nf, 1)
    rng = np.random.default_rng(seed)
    masks = rng.choice(allm, min(len(allm), 60), replace=False)
    _knn_case(snaps, oracle_mod, X, masks, k, engine="grid")


def test_grid_engine_ties(snaps, oracle_mod):
    # candidates do not arrive in id order: ties at the threshold must still go to the smaller id
    X = workloads.hypercube_table(9)
    _knn_case(snaps, oracle_mod, X, workloads.all_masks(9, 1)[::7], 10, engine="grid")
    X = workloads.duplicate_block_table(900, 3, frac=0.3)
    masks = np.array([(1 << 13) | (1 << 14), (1 << 13) | 1, 0x7FFF, 1 << 14, (1 << 6) | 3], dtype=np.uint16)
    g, _ = _knn_case(snaps, oracle_mod, X, masks, 10, engine="grid")
    oi, od = oracle_mod.knn_selfjoin(X, masks, 10)
    zero = od[0, :, -1] == 0
    assert zero.sum() > 100 and (g["idx"][0][zero] == oi[0][zero]).all()


def test_grid_engine_negative_and_signed_zero_columns(snaps, oracle_mod):
    # the quantile bins order values with an order-preserving key: negative coordinates and -0.0 are legal
    X = workloads.make_table(2500, 17, cols=list(range(8)), outlier_frac=0.02) - np.float32(0.5)
    X[::7, 2] = np.float32(-0.0)
    X[1::7, 2] = np.float32(0.0)
    masks = np.array([0b101, 0b1100, 0b11111111, 0b100, 0b1000110], dtype=np.uint16)
    _knn_case(snaps, oracle_mod, X, masks, 10, engine="grid")
    _knn_case(snaps, oracle_mod, X, masks, 10, engine="lattice")


@pytest.mark.parametrize("k", [33, 64, 256])
def test_grid_engine_large_k(snaps, oracle_mod, k):
    # NEXT-3: k beyond the sub-lattice engine's 32 (k_max = 256 on LSST5M); auto picks the grid engine
    X = workloads.make_table(1800, 19, cols=list(range(10)), outlier_frac=0.01)
    masks = np.array([0b11, 0b1010101, 0b1111111111, 0b1000000100, 0b110110], dtype=np.uint16)
    _knn_case(snaps, oracle_mod, X, masks, k)


def test_engines_agree(snaps, oracle_mod):
    # same joins from both engines: ids equal wherever the oracle says the query is unambiguous
    import torch
    X = workloads.make_table(4000, 13, outlier_frac=0.01)
    masks = workloads.pair_masks_plus_full(15)
    Xd = _dev(X)
    a = snaps.knn_selfjoin(Xd, masks, 10, engine="lattice")
    b = snaps.knn_selfjoin(Xd, masks, 10, engine="grid")
    torch.cuda.synchronize()
    same = (a["idx"] == b["idx"]).all(dim=2)
    assert same.float().mean().item() > 0.999
    assert torch.allclose(a["dist"], b["dist"], rtol=2e-6, atol=0)
    assert bool((a["indeg"].sum(dim=1) == b["indeg"].sum(dim=1)).all())


def test_query_range_slices_concatenate(snaps, oracle_mod):
    # a rank owns a query slice; slices concatenate, in-degree rows add
    import torch
    X = workloads.make_table(2600, 29, cols=list(range(12)), outlier_frac=0.01)
    masks = workloads.all_masks(12)[::41]
    Xd = _dev(X)
    for engine in ("lattice", "grid"):
        full = snaps.knn_selfjoin(Xd, masks, 9, engine=engine)
        cuts = [0, 700, 701, 1999, 2600]
        parts = [snaps.knn_selfjoin(Xd, masks, 9, engine=engine, q_range=(cuts[i], cuts[i + 1])) for i in range(4)]
        torch.cuda.synchronize()
        for n in ("idx", "dist", "kth", "mean"):
            assert torch.equal(torch.cat([p[n] for p in parts], dim=1), full[n]), (engine, n)
        assert torch.equal(sum(p["indeg"] for p in parts), full["indeg"]), engine
        eps = np.full(len(masks), 0.2, np.float32)
        rf = snaps.range_selfjoin(Xd, masks, eps, engine=engine)
        rp = [snaps.range_selfjoin(Xd, masks, eps, engine=engine, q_range=(cuts[i], cuts[i + 1])) for i in range(4)]
        torch.cuda.synchronize()
        assert torch.equal(torch.cat([p["count"] for p in rp], dim=1), rf["count"]), engine
        # the grid engine adds a query's distances in scan order, which depends on the 32 queries it is grouped with
        cat = torch.cat([p["sumdist"] for p in rp], dim=1)
        assert torch.equal(cat, rf["sumdist"]) if engine == "lattice" else torch.allclose(cat, rf["sumdist"], rtol=2e-5, atol=0)


def test_config4_full_size_sampled(snaps, oracle_mod):
    """BASELINE.json configs[3] at full size: N=1,000,000 x 15 (seed 3, 0.1% outliers), the 105
    two-feature subspaces plus the full space, k=10, lists and scores batched through pinned host
    memory.  The library takes the grid engine at this N.  All masks x 64 sampled queries against the oracle."""
    import torch
    cfg = workloads.get_config("c4_lsst_pairs")
    X, masks, k = cfg.table(), cfg.masks(), cfg.k
    n = len(X)
    st = snaps.knn_selfjoin_streamed(_dev(X), masks, k, masks_per_batch=16, lists=True)
    torch.cuda.synchronize()
    rng = np.random.default_rng(9)
    qs = np.sort(rng.choice(n, 64, replace=False))
    sel = np.arange(len(masks))                                  # all 106 masks
    oi, od = oracle_mod.knn_selfjoin(X, masks[sel], k + 1, queries=qs)
    check_knn(st["idx"][sel][:, qs].numpy(), st["dist"][sel][:, qs].numpy(), oi, od, queries=qs)
    kth = st["kth"][sel][:, qs].numpy().astype(np.float64)
    assert (np.abs(kth - od[:, :, k - 1]) <= 1e-4 * od[:, :, k - 1] + 1e-7).all()
    assert bool((st["indeg"].sum(dim=1) == n * k).all())


@pytest.mark.parametrize("n,nf,seed", [(2, 2, 0), (130, 5, 1), (1537, 15, 3), (3000, 15, 5)])
def test_grid_engine_range_join(snaps, oracle_mod, n, nf, seed):
    import torch
    X = workloads.make_table(n, seed, cols=list(range(nf)), outlier_frac=0.02)
    allm = workloads.all_masks(nf, 1)
    rng = np.random.default_rng(seed)
    masks = rng.choice(allm, min(len(allm), 48), replace=False)
    _, od = oracle_mod.knn_selfjoin(X, masks, min(10, n - 1))
    eps = np.array([max(1.003 * np.median(od[m, :, -1]), 1e-3) for m in range(len(masks))], dtype=np.float32)
    out = snaps.range_selfjoin(_dev(X), masks, eps, engine="grid")
    torch.cuda.synchronize()
    lo, hi = check_range(out["count"].cpu().numpy(), out["sumdist"].cpu().numpy(), out["mean"].cpu().numpy(),
                         oracle_mod, X, masks, eps)
    assert (lo == hi).mean() > 0.99


def test_eps_grid_by_repeating_masks(snaps, oracle_mod):
    """The eps grid of PAPER.md:181 through the existing entry point: a mask listed once per radius.
    Result sets are nested, A(eps_1) within A(eps_2) within A(eps_3) (Fig. 3)."""
    import torch
    X = workloads.make_table(1500, 23, outlier_frac=0.01)
    base = np.array([0b11, 0x7FFF, (1 << 7) | (1 << 2) | 1, 0b111100], dtype=np.uint16)
    grid = np.array([0.02, 0.05, 0.11], dtype=np.float32)
    masks = np.repeat(base, len(grid))
    eps = np.tile(grid, len(base)) * np.repeat(np.array([1.0, 6.0, 2.0, 3.0], dtype=np.float32), len(grid))
    out = snaps.range_selfjoin(_dev(X), masks, eps)
    torch.cuda.synchronize()
    cnt = out["count"].cpu().numpy()
    check_range(cnt, out["sumdist"].cpu().numpy(), out["mean"].cpu().numpy(), oracle_mod, X, masks, eps)
    c = cnt.reshape(len(base), len(grid), -1)
    assert (np.diff(c, axis=1) >= 0).all() and (c[:, -1] > c[:, 0]).any()


def test_config5_real_mask_list(snaps, oracle_mod):
    """BASELINE.json configs[4]'s own mask list (256 masks sampled from the 32,752, seed 4; 2-12 features),
    k=16 kNNSJ + DSSJ (~100 neighbours), outputs through the recycling sink (two pinned host buffers), at
    N=1,000,000 (the full N=5,000,000 pass takes minutes: `python bench.py --config c5_lsst_oversub`).
    Sampled (mask, query) rows of EVERY mask against the oracle; in-degree sums over every mask."""
    import torch
    cfg = workloads.get_config("c5_lsst_oversub")
    n, k = 1_000_000, cfg.k
    X = workloads.make_table(n, cfg.seed, outlier_frac=0.001)
    masks = cfg.masks()
    assert len(masks) == 256 and workloads.popcount(masks).max() >= 10
    Xd = _dev(X)
    rng = np.random.default_rng(3)
    qs = np.sort(rng.choice(n, 8, replace=False))
    got = {"idx": np.empty((256, 8, k), np.int32), "dist": np.empty((256, 8, k), np.float32),
           "kth": np.empty((256, 8), np.float32), "indeg_sum": np.zeros(256, np.int64), "groups": 0}

    def consume(m0, m1, a):
        got["idx"][m0:m1] = a["idx"][:, qs]
        got["dist"][m0:m1] = a["dist"][:, qs]
        got["kth"][m0:m1] = a["kth"][:, qs]
        got["indeg_sum"][m0:m1] = a["indeg"].sum(axis=1, dtype=np.int64)
        got["groups"] += 1

    ws = snaps.knn_selfjoin_sink(Xd, masks, k, 6, consume, want=("idx", "dist", "kth", "indeg"))
    assert got["groups"] == (256 + 5) // 6
    oi, od = oracle_mod.knn_selfjoin(X, masks, k + 1, queries=qs)
    check_knn(got["idx"], got["dist"], oi, od, queries=qs)
    assert (np.abs(got["kth"] - od[:, :, k - 1]) <= 1e-4 * od[:, :, k - 1] + 1e-7).all()
    assert (got["indeg_sum"] == n * k).all()                        # PAPER.md:136, every mask
    # DSSJ: radii from the library's own search (NEXT-2) for ~100 neighbours, then the join through the sink
    eps = snaps.eps_for_selectivity(Xd, masks, cfg.target_neighbours, seed=cfg.seed)
    r = {"count": np.empty((256, 8), np.uint32), "sumdist": np.empty((256, 8), np.float32),
         "mean": np.empty((256, 8), np.float32), "total": 0}

    def consume_r(m0, m1, a):
        r["count"][m0:m1] = a["count"][:, qs]
        r["sumdist"][m0:m1] = a["sumdist"][:, qs]
        r["mean"][m0:m1] = a["eps_mean"][:, qs]
        r["total"] += int(a["count"].sum(dtype=np.int64))

    snaps.range_selfjoin_sink(Xd, masks, eps, 6, consume_r, workspace=ws)
    check_range(r["count"], r["sumdist"], r["mean"], oracle_mod, X, masks, eps, queries=qs)
    assert 30 < r["total"] / (256.0 * n) < 300                      # the search aimed at ~100 neighbours


def test_sink_matches_resident(snaps, oracle_mod):
    # the recycling sink hands out exactly what the resident call writes, group by group, both engines
    import torch
    X = workloads.make_table(1500, 37, cols=list(range(11)))
    masks = workloads.all_masks(11)[::13]
    Xd = _dev(X)
    for engine in ("lattice", "grid"):
        ref = snaps.knn_selfjoin(Xd, masks, 9, engine=engine)
        rr = snaps.range_selfjoin(Xd, masks, np.full(len(masks), 0.15, np.float32), engine=engine)
        torch.cuda.synchronize()
        seen = []

        def consume(m0, m1, a):
            seen.append((m0, m1))
            for n in ("idx", "dist", "kth", "mean", "indeg"):
                assert (a[n] == ref[n][m0:m1].cpu().numpy()).all(), (engine, n)

        snaps.knn_selfjoin_sink(Xd, masks, 9, 7, consume, want=("idx", "dist", "kth", "mean", "indeg"), n_buffers=3,
                                engine=engine)
        assert seen == [(m, min(m + 7, len(masks))) for m in range(0, len(masks), 7)]

        def consume_r(m0, m1, a):
            assert (a["count"] == rr["count"][m0:m1].cpu().numpy().view(np.uint32)).all()
            assert (a["sumdist"] == rr["sumdist"][m0:m1].cpu().numpy()).all()
            assert (a["eps_mean"] == rr["mean"][m0:m1].cpu().numpy()).all()

        snaps.range_selfjoin_sink(Xd, masks, np.full(len(masks), 0.15, np.float32), 5, consume_r, engine=engine)


# ---------------------------------------------------------------- NEXT-3: the paper's operating points
@pytest.mark.parametrize("k", [64, 256])
def test_paper_operating_point_large_k(snaps, oracle_mod, k):
    """PAPER.md:440 (LSST5M: k_max = 256) on the SNAPShot1-shaped table: N = 31,693, 64 masks stratified over
    d = 2..15, k = 64 and 256 (the grid engine; the sub-lattice engine stops at 32).  Sampled queries of every
    mask against the oracle, in-degree sums over the whole output."""
    import torch
    cfg = workloads.get_config("c2_snapshot1_knn")
    X, allm = cfg.table(), cfg.masks()
    N = len(X)
    rng = np.random.default_rng(k)
    pc = workloads.popcount(allm)
    masks = allm[np.sort(np.concatenate([rng.choice(np.flatnonzero(pc == d), min(5, int((pc == d).sum())), replace=False)
                                         for d in range(2, 16)]))][:64]
    out = snaps.knn_selfjoin(_dev(X), masks, k)
    torch.cuda.synchronize()
    qs = np.sort(rng.choice(N, 12, replace=False))
    oi, od = oracle_mod.knn_selfjoin(X, masks, k + 1, queries=qs)
    check_knn(out["idx"][:, qs].cpu().numpy(), out["dist"][:, qs].cpu().numpy(), oi, od, queries=qs)
    kth = out["kth"][:, qs].cpu().numpy().astype(np.float64)
    assert (np.abs(kth - od[:, :, k - 1]) <= 1e-4 * od[:, :, k - 1] + 1e-7).all()
    assert bool((out["indeg"].sum(dim=1) == N * k).all())


def test_paper_operating_point_large_selectivity(snaps, oracle_mod):
    """PAPER.md:229 (s_min ~ 0.001 |D|, s_max ~ 0.15 |D| ~ 4,754 neighbours on SNAPShot1): the radius grid from
    eps_min to eps_max in ONE scan through the grid engine at N = 31,693; radii from the
    library's own search; sampled queries of every radius against the oracle evaluated once per radius."""
    import torch
    cfg = workloads.get_config("c3_snapshot1_dssj")
    X = cfg.table()
    N = len(X)
    masks = np.array([0b11, (1 << 9) | (1 << 3) | 1, 0b1111000, 0x7FFF, (1 << 14) | (1 << 7) | (1 << 6) | (1 << 2)], dtype=np.uint16)
    rng = np.random.default_rng(17)
    q = np.sort(rng.choice(N, 400, replace=False))
    c = np.sort(rng.choice(N, 8000, replace=False))
    es = snaps.eps_search(_dev(X), masks, q, c, [0.001 * N, 0.15 * N], 2048)["eps"].cpu().numpy()
    G = 6
    grid = np.stack([np.linspace(es[m, 0], es[m, 1], G, dtype=np.float32) for m in range(len(masks))])
    out = snaps.range_selfjoin_grid(_dev(X), masks, grid, engine="grid")
    torch.cuda.synchronize()
    qs = np.sort(rng.choice(N, 10, replace=False))
    for g in range(G):
        check_range(out["count"][:, g][:, qs].cpu().numpy(), out["sumdist"][:, g][:, qs].cpu().numpy(),
                    out["mean"][:, g][:, qs].cpu().numpy(), oracle_mod, X, masks, grid[:, g], queries=qs)
    mean_cnt = out["count"].float().mean(dim=2).cpu().numpy()
    assert (mean_cnt[:, 0] > 0.0003 * N).all() and (mean_cnt[:, 0] < 0.004 * N).all()      # ~0.001 |D|
    assert (mean_cnt[:, -1] > 0.08 * N).all() and (mean_cnt[:, -1] < 0.3 * N).all()         # ~0.15 |D|


def test_paper_operating_point_k4096(snaps, oracle_mod):
    """k_max = 4096 on SNAPShot1 (13 % of the catalogue).  N = 31,693, three masks, k = 4096: the
    grid engine with its heaps in the output lists.  Sampled queries against the oracle; whole-output invariants."""
    import torch
    cfg = workloads.get_config("c2_snapshot1_knn")
    X = cfg.table()
    N, k = len(X), 4096
    masks = np.array([0b11, (1 << 9) | (1 << 3) | 1 | (1 << 12), 0x7FFF], dtype=np.uint16)
    out = snaps.knn_selfjoin(_dev(X), masks, k)
    torch.cuda.synchronize()
    rng = np.random.default_rng(4096)
    qs = np.sort(rng.choice(N, 6, replace=False))
    oi, od = oracle_mod.knn_selfjoin(X, masks, k + 1, queries=qs)
    check_knn(out["idx"][:, qs].cpu().numpy(), out["dist"][:, qs].cpu().numpy(), oi, od, queries=qs)
    assert bool((out["indeg"].sum(dim=1) == N * k).all())
    assert bool((out["dist"][:, :, 1:] >= out["dist"][:, :, :-1]).all())
    assert torch.equal(out["kth"], out["dist"][:, :, -1])


@pytest.mark.parametrize("n,nf,k,seed", [(700, 15, 385, 0), (1200, 6, 1000, 1), (1537, 15, 700, 2), (600, 3, 599, 3)])
def test_long_list_path_against_oracle(snaps, oracle_mod, n, nf, k, seed):
    """k > 384 on a small table takes the selection path (knn_bigk.cu: radix selection over brute-force passes,
    then one segmented sort): whole output against the oracle, incl. k = N - 1, plus a table with a block of
    duplicate rows (every tie must go to the smaller id) and a query-range slice."""
    import torch
    X = workloads.make_table(n, 50 + seed, cols=list(range(nf)), outlier_frac=0.02)
    if seed == 2:
        X = workloads.duplicate_block_table(n, 50 + seed)
    allm = workloads.all_masks(nf, 1)
    masks = np.random.default_rng(seed).choice(allm, 5, replace=False).astype(np.uint16)
    g, _ = _knn_case(snaps, oracle_mod, X, masks, k, engine="grid")
    # a slice of the queries gives the same rows
    q0, q1 = n // 3, n // 3 + 101
    part = snaps.knn_selfjoin(_dev(X), masks, k, engine="grid", q_range=(q0, q1))
    torch.cuda.synchronize()
    assert np.array_equal(part["idx"].cpu().numpy(), g["idx"][:, q0:q1])
    assert np.array_equal(part["dist"].cpu().numpy(), g["dist"][:, q0:q1])
    assert np.array_equal(part["mean"].cpu().numpy(), g["mean"][:, q0:q1])


def test_long_list_path_above_65535_objects(snaps, oracle_mod):
    """N >= 65,536: the selection path counts in 32 bits (a histogram bin can hold more than 65,535 candidates).
    Sampled queries against the oracle, whole-output invariants."""
    import torch
    N, k = 70001, 600
    X = workloads.make_table(N, 66, outlier_frac=0.001)
    masks = np.array([0b11, (1 << 12) | (1 << 8) | (1 << 3) | 1, 0x7FFF], dtype=np.uint16)
    out = snaps.knn_selfjoin(_dev(X), masks, k, engine="grid")
    torch.cuda.synchronize()
    qs = np.sort(np.random.default_rng(6).choice(N, 6, replace=False))
    oi, od = oracle_mod.knn_selfjoin(X, masks, k + 1, queries=qs)
    check_knn(out["idx"][:, qs].cpu().numpy(), out["dist"][:, qs].cpu().numpy(), oi, od, queries=qs)
    assert bool((out["indeg"].sum(dim=1) == N * k).all())
    assert bool((out["dist"][:, :, 1:] >= out["dist"][:, :, :-1]).all())
    assert torch.equal(out["kth"], out["dist"][:, :, -1])


def test_long_list_path_through_the_batched_calls(snaps):
    """Long lists through the streamed call (staging ring + side-stream copies) and through a query-range slice of
    it: the same outputs as the resident call."""
    import torch
    X = workloads.make_table(1800, 93, outlier_frac=0.01)
    masks = np.array([0b101, 0x7FFF, (1 << 9) | (1 << 2), 0b1111000, (1 << 14) | 1], dtype=np.uint16)
    k = 450
    Xd = _dev(X)
    ref = snaps.knn_selfjoin(Xd, masks, k, engine="grid")
    st = snaps.knn_selfjoin_streamed(Xd, masks, k, masks_per_batch=2, engine="grid")
    part = snaps.knn_selfjoin_streamed(Xd, masks, k, masks_per_batch=3, engine="grid", q_range=(500, 1301))
    torch.cuda.synchronize()
    for name in ("idx", "dist", "kth", "mean", "indeg"):
        assert torch.equal(st[name], ref[name].cpu()), name
    for name in ("idx", "dist", "kth", "mean"):
        assert torch.equal(part[name], ref[name][:, 500:1301].cpu()), name


def test_long_list_path_equals_heap_path(snaps):
    """The two ways of building lists longer than 256 give identical outputs: a workspace without the selection
    path's scratch (the size for k = 384) makes the same call fall back to the heaps in the output lists."""
    import torch
    X = workloads.make_table(2500, 91, outlier_frac=0.01)
    masks = np.array([0b11, 0x7FFF, (1 << 10) | (1 << 5) | 0b100], dtype=np.uint16)
    k = 777
    Xd = _dev(X)
    a = snaps.knn_selfjoin(Xd, masks, k, engine="grid")
    small = torch.empty(snaps.workspace_bytes(len(X), 15, len(masks), 384, engine="grid"), dtype=torch.uint8, device="cuda")
    assert small.numel() < a["_workspace"].numel()
    b = snaps.knn_selfjoin(Xd, masks, k, engine="grid", workspace=small)
    torch.cuda.synchronize()
    for name in ("idx", "dist", "kth", "mean", "indeg"):
        assert torch.equal(a[name], b[name]), name


def test_radius_grid_sub_lattice_engine_full_size(snaps, oracle_mod):
    """The sub-lattice radius-grid kernel (range_grid.cu) at config 3's size: N = 31,693, two whole batches
    (128 lattice slots, 125 masks), four radii per mask up to config 3's stored eps_d; sampled queries of every
    (mask, radius) against the oracle, and the largest radius against the single-radius kernel."""
    import torch
    cfg = workloads.get_config("c3_snapshot1_dssj")
    X, allm = cfg.table(), cfg.masks()
    N = len(X)
    hi = allm.astype(np.int64) >> 6
    masks = allm[np.isin(hi, [0, 0b100100001])]
    eps = workloads.config_eps(cfg.name, masks)
    grid = (eps[:, None] * np.array([0.4, 0.6, 0.8, 1.0], dtype=np.float32)[None, :]).astype(np.float32)
    Xd = _dev(X)
    out = snaps.range_selfjoin_grid(Xd, masks, grid, engine="lattice")
    one = snaps.range_selfjoin(Xd, masks, grid[:, -1].copy(), engine="lattice")
    torch.cuda.synchronize()
    assert torch.equal(out["count"][:, -1], one["count"])
    rng = np.random.default_rng(21)
    qs = np.sort(rng.choice(N, 8, replace=False))
    for g in range(grid.shape[1]):
        check_range(out["count"][:, g][:, qs].cpu().numpy(), out["sumdist"][:, g][:, qs].cpu().numpy(),
                    out["mean"][:, g][:, qs].cpu().numpy(), oracle_mod, X, masks, grid[:, g], queries=qs)
    assert bool((out["count"][:, 1:] >= out["count"][:, :-1]).all())          # nested result sets
