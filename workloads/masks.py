"""Feature-subspace bitmask lists (uint16, bit j <-> column j)."""
from __future__ import annotations

import numpy as np


def popcount(m) -> np.ndarray:
    m = np.asarray(m, dtype=np.uint32)
    c = np.zeros(m.shape, dtype=np.int32)
    for b in range(16):
        c += ((m >> b) & 1).astype(np.int32)
    return c


def all_masks(n_feat: int, min_dim: int = 2) -> np.ndarray:
    """Every subset of n_feat features with at least min_dim of them, in
    increasing numeric order (Eq. 1: 32,752 for n_feat=15)."""
    m = np.arange(1, 1 << n_feat, dtype=np.uint32)
    return m[popcount(m) >= min_dim].astype(np.uint16)


def pair_masks_plus_full(n_feat: int = 15) -> np.ndarray:
    """The C(n_feat,2) two-feature subspaces plus the full space (config 4)."""
    out = [(1 << a) | (1 << b) for a in range(n_feat) for b in range(a + 1, n_feat)]
    out.append((1 << n_feat) - 1)
    return np.array(out, dtype=np.uint16)


def sample_masks(n_masks: int, seed: int, n_feat: int = 15) -> np.ndarray:
    """n_masks drawn without replacement from all_masks(n_feat) (config 5)."""
    pool = all_masks(n_feat)
    rng = np.random.default_rng(seed)
    return np.sort(rng.choice(pool, n_masks, replace=False)).astype(np.uint16)
