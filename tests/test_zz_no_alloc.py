"""snaps_knn_selfjoin_static: the kNN self-join with the library's built-in scratch array (no
workspace, no device allocation in the call) against the existing workspace path -- the same kernels,
so the outputs are compared exactly -- on two calls in a row that share the scratch array.

Collected last (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

import workloads

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


def _outputs(snaps, X, masks, k):
    """Preallocated outputs, filled with a pattern the join must overwrite."""
    import torch
    n, N = len(masks), len(X)
    dev = torch.device("cuda")
    return {"idx": torch.full((n, N, k), -7, dtype=torch.int32, device=dev),
            "dist": torch.full((n, N, k), -7.0, dtype=torch.float32, device=dev),
            "kth": torch.full((n, N), -7.0, dtype=torch.float32, device=dev),
            "mean": torch.full((n, N), -7.0, dtype=torch.float32, device=dev),
            "indeg": torch.full((n, N), -7, dtype=torch.int32, device=dev)}


def _compare(snaps, X, masks, k):
    import torch
    Xd = _dev(X)
    out = _outputs(snaps, X, masks, k)
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    got = snaps.knn_selfjoin_static(Xd, masks, k, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before      # the wrapper was given every output
    ref = snaps.knn_selfjoin(Xd, masks, k, engine="lattice")
    torch.cuda.synchronize()
    for name in ("idx", "dist", "kth", "mean", "indeg"):
        a, b = got[name].cpu().numpy(), ref[name].cpu().numpy()
        assert np.array_equal(a, b), name
    N = len(X)
    assert (got["indeg"].sum(dim=1) == N * k).all()     # every object has k neighbours
    return got


def test_static_scratch_two_calls_in_a_row(snaps):
    # first call: several tiles, a ragged tail, masks from many batches
    X1 = workloads.make_table(3001, 11)
    all_masks = workloads.all_masks(15)
    rng = np.random.default_rng(5)
    m1 = np.sort(rng.choice(all_masks, 300, replace=False)).astype(np.uint16)
    g1 = _compare(snaps, X1, m1, 10)
    # second call right after it: a smaller table, fewer features, another k -- whatever the first call
    # left in the scratch array beyond the new sizes must not matter
    X2 = workloads.make_table(777, 12, cols=[0, 1, 3, 4, 5, 7, 9])
    m2 = workloads.all_masks(7)
    g2 = _compare(snaps, X2, m2, 7)
    assert g2["idx"].shape == (len(m2), 777, 7)
    # and the first inputs again: the same result as before
    g3 = _compare(snaps, X1, m1, 10)
    assert np.array_equal(g1["idx"].cpu().numpy(), g3["idx"].cpu().numpy())


def test_static_scratch_limits(snaps):
    import torch
    X = torch.zeros((snaps.STATIC_MAX_N + 1, 2), dtype=torch.float32, device="cuda")
    with pytest.raises(snaps.SnapsError, match="limit of the built-in scratch"):
        snaps.knn_selfjoin_static(X, np.array([3], np.uint16), 2, lists=False)
    Xs = _dev(workloads.make_table(64, 0))
    too_many = np.resize(workloads.all_masks(15), snaps.STATIC_MAX_MASKS + 1).astype(np.uint16)
    with pytest.raises(snaps.SnapsError, match="limit of the built-in scratch"):
        snaps.knn_selfjoin_static(Xs, too_many, 2, lists=False)
    with pytest.raises(snaps.SnapsError, match="k = 33"):
        snaps.knn_selfjoin_static(Xs, np.array([3], np.uint16), 33, lists=False)
