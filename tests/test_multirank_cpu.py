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
