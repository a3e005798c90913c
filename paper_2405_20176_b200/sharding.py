"""Multi-GPU sharding of one catalogue's mask list (host logic, no device work).

The method has no exchange step (feature spaces are independent and are dealt to the
least loaded GPU), so ranks share nothing but the replicated table.  Masks are dealt by *batch*
(all masks with the same features 6..14 stay together, so each rank still enumerates complete
sub-lattices and the per-pair squared differences are reused as on one GPU); batches are dealt
round-robin in Gray order so that every rank gets the same mix of subspace dimensions.
Outputs of the ranks concatenate; `unshard` gives the permutation back to the caller's order.
"""
from __future__ import annotations

import numpy as np

LOW_BITS = 6  # lattice features of a batch (csrc/snaps_device.cuh: kLow)


def _gray_rank(g: np.ndarray) -> np.ndarray:
    b = g.copy()
    s = 1
    while s < 16:
        b ^= b >> s
        s <<= 1
    return b


def shard_masks(masks, rank: int, world: int):
    """-> (indices into `masks` owned by `rank`, ascending).  Disjoint over ranks, covers all."""
    m = np.asarray(masks, dtype=np.uint16).astype(np.int64)
    assert 0 <= rank < world
    high = m >> LOW_BITS
    keys = np.unique(high)
    order = keys[np.argsort(_gray_rank(keys), kind="stable")]        # batches in Gray order
    owner = {int(h): i % world for i, h in enumerate(order)}
    mine = np.fromiter((owner[int(h)] == rank for h in high), dtype=bool, count=len(m))
    return np.flatnonzero(mine)


def unshard(index_lists, n_masks: int) -> np.ndarray:
    """Given every rank's index list, the permutation p with concat(outputs)[p] in caller order."""
    cat = np.concatenate(index_lists)
    assert len(cat) == n_masks and len(np.unique(cat)) == n_masks
    return np.argsort(cat, kind="stable")


def shard_queries(n_objects: int, rank: int, world: int):
    """-> (q_begin, q_end): the contiguous slice of query ids `rank` owns (table
    replicated, every rank joins its slice against all objects; lists and scores concatenate in rank
    order, the in-degree rows of the ranks add up)."""
    assert 0 <= rank < world
    return n_objects * rank // world, n_objects * (rank + 1) // world


def shard_masks_by_cost(masks, rank: int, world: int):
    """Grid engine (one subspace per launch, cost grows with the number of features): masks sorted by
    popcount and dealt round-robin, so that every rank gets the same mix.  -> indices, ascending."""
    m = np.asarray(masks, dtype=np.uint16).astype(np.int64)
    assert 0 <= rank < world
    pc = np.zeros(len(m), dtype=np.int64)
    for b in range(16):
        pc += (m >> b) & 1
    order = np.argsort(pc, kind="stable")
    return np.sort(order[rank::world])


def mask_groups(masks, batches_per_group: int = 8):
    """The mask list cut into groups of whole sub-lattice batches in Gray order (the unit of work a rank
    takes at a time under dynamic dealing).  -> list of index arrays into `masks`."""
    m = np.asarray(masks, dtype=np.uint16).astype(np.int64)
    high = m >> LOW_BITS
    keys = np.unique(high)
    order = keys[np.argsort(_gray_rank(keys), kind="stable")]
    groups = []
    for g0 in range(0, len(order), batches_per_group):
        sel = np.isin(high, order[g0:g0 + batches_per_group])
        groups.append(np.flatnonzero(sel))
    return groups


class DynamicDealer:
    """"the least loaded GPU is assigned the next feature space".  A shared counter in the
    job's torch.distributed store hands out work-unit indices in order: a rank that finishes early simply
    takes the next unit.  No data-path collective; the only traffic is one integer per unit."""

    def __init__(self, store, n_units: int, name: str = "snaps_next_unit"):
        self.store, self.n_units, self.name = store, n_units, name

    def __iter__(self):
        while True:
            unit = int(self.store.add(self.name, 1)) - 1
            if unit >= self.n_units:
                return
            yield unit
