"""Writes workloads/config_eps.json: the per-dimension radii eps_d of the DSSJ configurations
(BASELINE.json configs[2]: "eps_d computed by the oracle on a 1,000-point sample" for a mean of
~50 neighbours) -- TEST INFRASTRUCTURE.  Calls only oracle/ and the seeded generators; bench.py and
the library read the stored numbers as INPUTS and never import oracle/ for them.

    python -m oracle.write_config_eps
"""
from __future__ import annotations

import json
import os

import numpy as np

import workloads
from oracle.calibrate import eps_per_dimension


def main():
    out = {}
    for name in ("c3_snapshot1_dssj",):
        cfg = workloads.get_config(name)
        X, masks = cfg.table(), cfg.masks()
        eps = eps_per_dimension(X, masks, cfg.target_neighbours, seed=cfg.seed, max_masks_per_dim=4,
                                n_query_sample=300)
        dims = workloads.popcount(masks)
        out[name] = {"target_neighbours": cfg.target_neighbours,
                     "recipe": "oracle.calibrate.eps_per_dimension(seed=cfg.seed, max_masks_per_dim=4, "
                               "n_query_sample=300) on the rank-0 table",
                     "eps_by_dimension": {str(int(d)): float(np.float32(eps[dims == d][0])) for d in np.unique(dims)}}
    path = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "workloads", "config_eps.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
