"""Synthetic asteroid feature tables shaped like SNAPShot1 / LSST5M.

The real tables (sections 2.1-2.2) are not available; these
stand in for them.  Column distributions follow BASELINE.json configs[0..1] and
Table 1; every column is min-max normalised to [0, 1]
(section 3.3) and cast to fp32.
"""
from __future__ import annotations

import numpy as np

COLUMN_NAMES = [
    "rotper", "lcamp", "H", "a", "e", "i", "color0", "color1",
    "G0", "G1", "derived0", "derived1", "derived2", "derived3", "derived4",
]

# analytic medians of the inlier distributions (the "5x wider" stretch is about these)
_MEDIANS = [
    float(np.sqrt(2.0 * 1000.0)),          # log-uniform 2..1000
    float(np.exp(-1.5)),                   # lognormal mu=-1.5
    16.0,                                  # N(16, 1.5)
    2.8,                                   # U(2.1, 3.5)
    0.12579,                               # Beta(2, 12)
    float(6.0 * np.sqrt(2.0 * np.log(2.0))),  # Rayleigh sigma=6
    0.5, 0.5, 0.15, 0.15,
    0.0, 0.0, 0.0, 0.0, 0.0,
]

_CHOL = np.linalg.cholesky(0.7 * np.eye(5) + 0.3 * np.ones((5, 5)))


def _draw_column(rng: np.random.Generator, col: int, n: int) -> np.ndarray:
    if col == 0:
        return np.exp(rng.uniform(np.log(2.0), np.log(1000.0), n))
    if col == 1:
        return rng.lognormal(-1.5, 0.6, n)
    if col == 2:
        return rng.normal(16.0, 1.5, n)
    if col == 3:
        return rng.uniform(2.1, 3.5, n)
    if col == 4:
        return rng.beta(2.0, 12.0, n)
    if col == 5:
        return rng.rayleigh(6.0, n)
    if col in (6, 7):
        return rng.normal(0.5, 0.1, n)
    if col in (8, 9):
        return rng.normal(0.15, 0.05, n)
    raise ValueError(col)


def _draw_block(rng: np.random.Generator, cols: list[int], n: int) -> np.ndarray:
    """Inlier draws for `cols` (in the given order); the 5 derived columns are
    drawn jointly (correlation 0.3) when the first of them is reached."""
    out = np.empty((n, len(cols)), dtype=np.float64)
    derived = None
    for pos, c in enumerate(cols):
        if c >= 10:
            if derived is None:
                derived = rng.standard_normal((n, 5)) @ _CHOL.T
            out[:, pos] = derived[:, c - 10]
        else:
            out[:, pos] = _draw_column(rng, c, n)
    return out


def make_table(n: int, seed: int, cols: list[int] | None = None,
               outlier_frac: float = 0.01) -> np.ndarray:
    """N x len(cols) fp32 table, C-contiguous, values in [0, 1], no NaN.

    Draw order (fixed): inlier columns in column order -> outlier row set ->
    fresh inlier draws for those rows, stretched 5x about the column median ->
    per-column min-max in fp64 -> fp32.
    """
    cols = list(range(15)) if cols is None else list(cols)
    rng = np.random.default_rng(seed)
    x = _draw_block(rng, cols, n)
    n_out = int(round(outlier_frac * n))
    if n_out > 0:
        rows = rng.choice(n, n_out, replace=False)
        v = _draw_block(rng, cols, n_out)
        med = np.array([_MEDIANS[c] for c in cols])
        x[rows, :] = med + 5.0 * (v - med)
    lo = x.min(axis=0)
    hi = x.max(axis=0)
    x = (x - lo) / (hi - lo)
    out = np.ascontiguousarray(x.astype(np.float32))
    assert not np.isnan(out).any() and out.min() == 0.0 and out.max() == 1.0
    return out


def hypercube_table(d: int) -> np.ndarray:
    """The 2^d vertices of {0,1}^d, row r = binary digits of r (bit j -> column j)."""
    r = np.arange(1 << d, dtype=np.int64)
    return np.ascontiguousarray(((r[:, None] >> np.arange(d)) & 1).astype(np.float32))


def lattice_table(n: int, n_feat: int, h: float, seed: int = 0) -> np.ndarray:
    """Column 0 is the 1-D lattice i*h (h a power of two keeps it exact);
    the other columns are random filler that a one-feature mask ignores."""
    rng = np.random.default_rng(seed)
    x = rng.random((n, n_feat)).astype(np.float32)
    x[:, 0] = (np.arange(n, dtype=np.float64) * h).astype(np.float32)
    return np.ascontiguousarray(x)


def duplicate_block_table(n: int, seed: int, frac: float = 0.3,
                          dup_cols: tuple[int, int] = (13, 14)) -> np.ndarray:
    """make_table() with `frac` of the rows sharing one value in two columns:
    the structure mean-imputation gives the two NEOWISE columns."""
    x = make_table(n, seed)
    rng = np.random.default_rng(seed + 1000)
    rows = rng.choice(n, int(round(frac * n)), replace=False)
    for c in dup_cols:
        x[rows, c] = np.float32(np.mean(x[:, c], dtype=np.float64))
    return np.ascontiguousarray(x)
