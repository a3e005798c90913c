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


def _knn_case(snaps, oracle_mod, X, masks, k, full_scores=True):
    import torch
    out = snaps.knn_selfjoin(_dev(X), masks, k)
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
        snaps.knn_selfjoin(X, [0b11], 33)                # k > SNAPS_MAX_K
    with pytest.raises(snaps.SnapsError):
        snaps.range_selfjoin(X, [0b11], [float("nan")])
    with pytest.raises(snaps.SnapsError):
        snaps.range_selfjoin(X, [0b11], [0.0])
    with pytest.raises(snaps.SnapsError) as e:
        snaps.knn_selfjoin(X, [0b11], 3, workspace=torch.empty(256, dtype=torch.uint8, device="cuda"))
    assert e.value.status == 3
    with pytest.raises(snaps.SnapsError):
        snaps.knn_selfjoin(X, [0b11], 3, lists=False, scores=False)
