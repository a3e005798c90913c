"""Pins for oracle/ranking.py against the paper's own worked examples (NEXT-1)."""
import os

import numpy as np

from oracle import ranking

HERE = os.path.dirname(os.path.abspath(__file__))


def _table2():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "table2_paper.txt"))
            if l.strip() and not l.startswith("#")]
    a = np.array(rows, dtype=np.float64)
    # point, dssj_count, rank, dssj_mean, rank, knn_indeg, rank, knn_mean, rank
    return a


def test_table2_ranks_from_table2_metrics():
    # PAPER.md:282-295 Table 2: every rank column follows from its metric column
    t = _table2()
    cnt, cnt_r, mean, mean_r, indeg, indeg_r, kmean, kmean_r = (t[:, i] for i in range(1, 9))
    assert ranking.dense_rank("dssj_count", cnt).tolist() == cnt_r.astype(int).tolist()
    assert ranking.dense_rank("dssj_mean", mean, counts=cnt).tolist() == mean_r.astype(int).tolist()
    assert ranking.dense_rank("knn_indegree", indeg).tolist() == indeg_r.astype(int).tolist()
    assert ranking.dense_rank("knn_mean", kmean).tolist() == kmean_r.astype(int).tolist()
    # point 10 is the only one with rank 0 in all four
    all0 = (cnt_r == 0) & (mean_r == 0) & (indeg_r == 0) & (kmean_r == 0)
    assert t[all0, 0].tolist() == [10.0]


def test_section_352_worked_example():
    rec = {}
    for l in open(os.path.join(HERE, "golden", "section352_example.txt")):
        if l.strip() and not l.startswith("#"):
            p = l.split()
            rec[p[0]] = [float(x) for x in p[1:]]
    sets = [np.array(rec[k], dtype=np.int64) for k in ("eps_1", "eps_2", "eps_3")]
    u_min, u_max = ranking.similarity_curves(sets, 10)
    assert u_min.tolist() == rec["U_min"] and u_max.tolist() == rec["U_max"]
    # Eq. 3: |U_min - U_max| = {0.8, 0.1, 0.8} -> the middle grid point is selected
    assert ranking.select_parameter(u_min, u_max) == 1


def test_topn_and_ties():
    v = np.array([3, 1, 1, 0, 2, 1])
    assert ranking.dense_rank("dssj_count", v).tolist() == [3, 1, 1, 0, 2, 1]
    assert ranking.topn_ids("dssj_count", v, 3).tolist() == [3, 1, 2]          # ties -> smaller id
    assert ranking.topn_ids("knn_mean", v.astype(float), 2).tolist() == [0, 4]  # largest first
    kth, mean, indeg = ranking.knn_scores_at_k(np.array([[1, 2, 0], [0, 2, 1], [1, 0, 2]])[:, :3],
                                               np.array([[1., 2., 3.], [1., 1., 4.], [2., 2., 2.]]), 2, 3)
    assert kth.tolist() == [2., 1., 2.] and mean.tolist() == [1.5, 1., 2.] and indeg.tolist() == [2, 2, 2]


def test_stored_config_eps_come_from_the_oracle_script():
    # workloads/config_eps.json is written by oracle/write_config_eps.py (calls only oracle/);
    # regenerate in memory and compare
    import workloads
    from oracle.calibrate import eps_per_dimension
    cfg = workloads.get_config("c3_snapshot1_dssj")
    X, masks = cfg.table(), cfg.masks()
    eps = eps_per_dimension(X, masks, cfg.target_neighbours, seed=cfg.seed, max_masks_per_dim=4,
                            n_query_sample=300).astype(np.float32)
    assert (workloads.config_eps(cfg.name, masks) == eps).all()
    assert (np.diff([eps[workloads.popcount(masks) == d][0] for d in range(2, 16)]) > 0).all()   # grows with d


def test_range_from_knn_is_the_range_join_where_complete():
    """oracle.ranking.range_from_knn against the oracle's own range join: wherever the k-th neighbour lies
    beyond eps, count / sum / mean read off the kNN list equal the eps-join's; elsewhere the
    count is the list length, a lower bound.  1-D lattice closed form on top: interior count = 2 floor(eps/h)."""
    import oracle
    import workloads
    from oracle.ranking import range_from_knn
    X = workloads.make_table(400, 5, cols=[0, 1, 2, 3])
    masks = np.array([0b11, 0b1111, 0b0110], dtype=np.uint16)
    k = 12
    _, od = oracle.knn_selfjoin(X, masks, k)
    for m in range(len(masks)):
        eps = float(np.median(od[m, :, 5]))          # about half the objects complete
        cnt, s, mean, complete = range_from_knn(od[m], eps)
        rc, rs, rm = oracle.range_selfjoin(X, masks[m:m + 1], [eps])
        assert 0.2 < complete.mean() < 0.9
        assert (cnt[complete] == rc[0][complete]).all() and np.allclose(s[complete], rs[0][complete], rtol=1e-12)
        assert np.allclose(mean[complete], rm[0][complete], rtol=1e-12)
        assert (cnt[~complete] == k).all() and (rc[0][~complete] >= k).all()
    h, n = 2.0 ** -6, 40
    L = workloads.lattice_table(n, 2, h)
    _, ld = oracle.knn_selfjoin(L, [0b01], 10)
    cnt, _, _, complete = range_from_knn(ld[0], 2.5 * h)
    assert (cnt[5:-5] == 4).all() and complete.all() and cnt[0] == 2
