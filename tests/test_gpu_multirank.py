"""Two ranks on two GPUs (skipped on a single-GPU box): the query-range sharding of SURVEY 8(e)(ii) through the
C ABI and NCCL -- each rank joins its slice of the queries, lists and scores are gathered in rank order, the
in-degree rows are all-reduced -- against the one-GPU join of the same catalogue, bit for bit."""
import os
import socket

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    import paper_2405_20176_b200 as snaps
    from paper_2405_20176_b200.sharding import shard_queries, shard_masks, unshard
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    torch.cuda.set_device(rank)
    dev = torch.device("cuda", rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    X = workloads.make_table(5000, 51, outlier_frac=0.01)
    masks = workloads.all_masks(15)[::517]
    Xd = torch.from_numpy(X).to(dev)
    k = 9
    for engine in ("lattice", "grid"):
        q0, q1 = shard_queries(len(X), rank, world)
        mine = snaps.knn_selfjoin(Xd, masks, k, q_range=(q0, q1), engine=engine)
        dist.all_reduce(mine["indeg"])                                   # the one exchange
        parts = [torch.empty((len(masks), shard_queries(len(X), r, world)[1] - shard_queries(len(X), r, world)[0], k),
                             dtype=torch.int32, device=dev) for r in range(world)]
        dist.all_gather(parts, mine["idx"].contiguous())
        full = snaps.knn_selfjoin(Xd, masks, k, engine=engine)
        torch.cuda.synchronize()
        assert torch.equal(torch.cat(parts, dim=1), full["idx"]), engine
        assert torch.equal(mine["indeg"], full["indeg"]), engine
    # masks dealt by batch: outputs concatenate and un-permute
    idx = shard_masks(masks, rank, world)
    part = snaps.knn_selfjoin(Xd, masks[idx], k, lists=False)["kth"]
    sizes = [len(shard_masks(masks, r, world)) for r in range(world)]
    bufs = [torch.empty((s, len(X)), dtype=torch.float32, device=dev) for s in sizes]
    dist.all_gather(bufs, part.contiguous())
    perm = unshard([shard_masks(masks, r, world) for r in range(world)], len(masks))
    whole = snaps.knn_selfjoin(Xd, masks, k, lists=False)["kth"]
    torch.cuda.synchronize()
    assert torch.equal(torch.cat(bufs)[torch.from_numpy(perm).to(dev)], whole)
    dist.barrier()
    dist.destroy_process_group()
    open(os.path.join(out_dir, f"gpu_ok{rank}"), "w").write("ok")


def test_two_gpus_query_ranges_and_mask_batches(tmp_path):
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    import torch.multiprocessing as mp
    mp.spawn(_worker, args=(2, _free_port(), str(tmp_path)), nprocs=2, join=True)
    assert all((tmp_path / f"gpu_ok{r}").exists() for r in range(2))
