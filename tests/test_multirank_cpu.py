"""World-size-2 gloo test (CPU) of the N>1 host logic: mask sharding by batch, the max-over-ranks
timing reduction of bench.py, and concatenation of per-rank outputs back into caller order."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2405_20176_b200.sharding import shard_masks, unshard
    masks = workloads.all_masks(15)
    mine = shard_masks(masks, rank, world)
    # every rank's shard keeps whole batches (same high bits never split over ranks)
    high_mine = set((masks[mine].astype(np.int64) >> 6).tolist())
    sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(sizes, torch.tensor([len(mine)], dtype=torch.int64))
    pad = int(max(s.item() for s in sizes))
    buf = torch.full((pad,), -1, dtype=torch.int64)
    buf[:len(mine)] = torch.from_numpy(mine)
    allidx = [torch.zeros(pad, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(allidx, buf)
    lists = [a[a >= 0].numpy() for a in allidx]
    cat = np.concatenate(lists)
    assert len(cat) == len(masks) and len(np.unique(cat)) == len(masks)          # disjoint cover
    for r, l in enumerate(lists):
        if r != rank:
            assert not (high_mine & set((masks[l].astype(np.int64) >> 6).tolist()))
    assert abs(len(lists[0]) - len(lists[1])) <= 64                               # balanced
    # a stand-in "score" per mask (its own value), produced per rank, concatenated, un-permuted
    outs = [masks[l].astype(np.int64) for l in lists]
    perm = unshard(lists, len(masks))
    assert (np.concatenate(outs)[perm] == masks.astype(np.int64)).all()
    # bench.py's timing rule: the step time of the job is the max over ranks
    t = torch.tensor([10.0 + rank], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    assert t.item() == 10.0 + world - 1
    dist.barrier()
    dist.destroy_process_group()
    open(os.path.join(out_dir, f"ok{rank}"), "w").write("ok")


def test_shard_masks_world2_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert all((tmp_path / f"ok{r}").exists() for r in range(world))


def test_shard_masks_single_process_properties():
    from paper_2405_20176_b200.sharding import shard_masks
    masks = workloads.sample_masks(256, 4)
    for world in (1, 3, 8):
        parts = [shard_masks(masks, r, world) for r in range(world)]
        cat = np.sort(np.concatenate(parts))
        assert (cat == np.arange(len(masks))).all()


def _query_worker(rank, world, port, out_dir):
    """SURVEY 8(e)(ii) on CPU: each rank owns the query slice `shard_queries` gives it; lists concatenate in
    rank order and the per-rank in-degree rows (histograms over the rank's own queries) add up to the
    full in-degree under one all-reduce -- the only exchange of query-range sharding.  The per-rank join
    is played by the oracle (the CUDA kernels need a GPU; their slice outputs are checked against the full
    join in tests/test_gpu_parity.py::test_query_range_slices_concatenate)."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_2405_20176_b200.sharding import shard_queries, shard_masks_by_cost
    n, k = 601, 5
    X = workloads.make_table(n, 21, cols=list(range(6)))
    masks = workloads.all_masks(6)[::5]
    q0, q1 = shard_queries(n, rank, world)
    idx, dist_ = oracle.knn_selfjoin(X, masks, k, queries=np.arange(q0, q1))
    indeg = np.stack([np.bincount(idx[m].ravel(), minlength=n) for m in range(len(masks))]).astype(np.int32)
    t = torch.from_numpy(indeg)
    dist.all_reduce(t)                                              # the in-degree sum over ranks
    sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(sizes, torch.tensor([q1 - q0], dtype=torch.int64))
    pad = int(max(s.item() for s in sizes))
    buf = torch.full((len(masks), pad, k), -1, dtype=torch.int32)
    buf[:, :q1 - q0] = torch.from_numpy(idx)
    parts = [torch.zeros_like(buf) for _ in range(world)]
    dist.all_gather(parts, buf)
    cat = torch.cat([p[:, :int(s.item())] for p, s in zip(parts, sizes)], dim=1).numpy()
    full_idx, full_dist = oracle.knn_selfjoin(X, masks, k)
    _, _, full_indeg = oracle.knn_scores(n, full_idx, full_dist)
    assert (cat == full_idx).all()                                  # slices concatenate in rank order
    assert (t.numpy() == full_indeg).all()                          # in-degree rows add up
    # slices are a disjoint cover; cost-balanced mask dealing is one too
    assert sum(int(s.item()) for s in sizes) == n
    m_all = np.sort(np.concatenate([shard_masks_by_cost(masks, r, world) for r in range(world)]))
    assert (m_all == np.arange(len(masks))).all()
    dist.barrier()
    dist.destroy_process_group()
    open(os.path.join(out_dir, f"q_ok{rank}"), "w").write("ok")


def test_query_range_sharding_world2_gloo(tmp_path):
    world = 2
    mp.spawn(_query_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert all((tmp_path / f"q_ok{r}").exists() for r in range(world))


def _dealer_worker(rank, world, port, out_dir):
    """Dynamic dealing: two ranks of different speed drain one counter; the units they take are a
    disjoint cover, and the slower rank ends up with fewer of them."""
    import time
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2405_20176_b200.sharding import DynamicDealer, mask_groups
    masks = workloads.all_masks(15)
    groups = mask_groups(masks, 8)
    assert len(groups) == 64 and sum(len(g) for g in groups) == len(masks)
    assert len(np.unique(np.concatenate(groups))) == len(masks)
    store = dist.distributed_c10d._get_default_store()
    dist.barrier()
    mine = []
    for unit in DynamicDealer(store, len(groups), name="t_units"):
        mine.append(unit)
        time.sleep(0.02 if rank == 0 else 0.002)              # rank 0 is the slow GPU
    got = [None] * world
    dist.all_gather_object(got, mine)
    allu = sorted(u for g in got for u in g)
    assert allu == list(range(len(groups)))
    assert len(got[0]) < len(got[1])
    dist.barrier()
    dist.destroy_process_group()
    open(os.path.join(out_dir, f"d_ok{rank}"), "w").write("ok")


def test_dynamic_dealing_world2_gloo(tmp_path):
    world = 2
    mp.spawn(_dealer_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert all((tmp_path / f"d_ok{r}").exists() for r in range(world))
