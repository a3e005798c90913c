"""Seeded randomised parity sweep: ragged N, every list stride (k up to 32), 1..15 features, heavy
ties and duplicated rows, repeated masks, both engines (sub-lattice / grid), kNN and range
joins -- each case element by element against the fp64 oracle under tests/parity.py's rules."""
import numpy as np
import pytest

import workloads
from parity import check_knn, check_knn_scores, check_range

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("seed", [11, 12, 13, 14])
def test_random_cases_against_oracle(seed, oracle_mod):
    import torch
    import paper_2405_20176_b200 as snaps
    rng = np.random.default_rng(seed)
    for case in range(40):
        nf = int(rng.integers(1, 16))
        n = int(rng.choice([2, 3, 31, 32, 33, 64, 65, 127, 500, 1024, 2047]))
        k = int(min(n - 1, rng.choice([1, 2, 5, 10, 12, 13, 16, 20, 21, 28, 29, 32])))
        kind = int(rng.integers(0, 4))
        if kind == 0:
            X = workloads.make_table(max(n, 3), int(rng.integers(1 << 30)), cols=list(range(nf)), outlier_frac=0.02)[:n]
        elif kind == 1:
            X = np.round(rng.random((n, nf)) * 4).astype(np.float32) / 4            # coarse grid: heavy ties
        elif kind == 2:
            X = rng.random((n, nf)).astype(np.float32)
            X[rng.random(n) < 0.4] = X[0]                                            # duplicates of row 0
        else:
            X = rng.random((n, nf)).astype(np.float32)
        X = np.ascontiguousarray(X)
        allm = workloads.all_masks(nf, 1)
        masks = rng.choice(allm, min(len(allm), int(rng.integers(1, 70))),
                           replace=bool(rng.integers(0, 2)) and len(allm) > 1)
        engine = ("lattice", "grid")[int(rng.integers(0, 2))]
        Xd = torch.from_numpy(X).cuda()
        out = snaps.knn_selfjoin(Xd, masks, k, engine=engine)
        torch.cuda.synchronize()
        g = {a: out[a].cpu().numpy() for a in ("idx", "dist", "kth", "mean", "indeg")}
        kk = min(k + 1, n - 1)
        oi, od = oracle_mod.knn_selfjoin(X, masks, kk)
        if kk == k:
            oi = np.concatenate([oi, np.full(oi.shape[:2] + (1,), -1, oi.dtype)], axis=2)
            od = np.concatenate([od, np.full(od.shape[:2] + (1,), np.inf)], axis=2)
        unamb = check_knn(g["idx"], g["dist"], oi, od)
        kth, mean, indeg = oracle_mod.knn_scores(n, oi[:, :, :k], od[:, :, :k])
        check_knn_scores(g, g["idx"], kth, mean, indeg, unamb, n)
        eps = np.maximum(np.median(od[:, :, k - 1], axis=1) * 1.00317, 1e-3).astype(np.float32)
        r = snaps.range_selfjoin(Xd, masks, eps, engine=engine)
        torch.cuda.synchronize()
        check_range(r["count"].cpu().numpy(), r["sumdist"].cpu().numpy(), r["mean"].cpu().numpy(),
                    oracle_mod, X, masks, eps)
