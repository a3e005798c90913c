#!/usr/bin/env python
"""bench.py -- all-subspace kNN self-join (BASELINE.json configs[1]) on N GPUs of one node.

A step = one pass of the whole hot path over one synthetic
SNAPShot1-shaped table: stage the N x 15 fp32 table, plan the 32,752 subspace masks into
sub-lattice batches, per-pair squared differences, add-only subset sums, per-(query, subspace)
top-k selection, and the fused per-object outlier scores (k-th distance, mean kNN distance,
kNN-graph in-degree).  `value` is timed with inputs resident in HBM; `e2e` is ONE C-ABI call with
host buffers (pinned table in, pinned scores out; both copies inside the timed region).

The default line also carries `dssj` (config 3: the eps range self-join over all 32,752 subspaces),
`lsst_scale` (config 4: N = 1,000,000 through the grid engine, outputs streamed to pinned host)
and `cpu_baseline` (the fp64 oracle on the host cores).  `--config c5_lsst_oversub` runs config 5
(N = 5,000,000, 256 sampled masks, kNN k=16 + DSSJ, outputs through the recycling sink).

Multi-GPU (`--gpus N` under torchrun): ONE catalogue, replicated; the mask list is dealt to the
ranks by sub-lattice batch (`sharding.shard_masks`), no data-path collective --
strong scaling.  `--scaling weak` gives every rank its own catalogue instead.  Configs 4-5 shard
by query range; the only exchange is the sum of the in-degree rows.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config NAME]
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "subspaces/sec and pair-distance evals/sec (kNNSJ N=31,693,k=10); % FP32 peak"
UNIT = "subspaces/s"
N_SM, LANES_PER_SM = 148, 128
KERNEL_SOURCES = ("paper_2405_20176_b200/csrc/knn_lattice.cu", "paper_2405_20176_b200/csrc/snaps_device.cuh")


def derived_peak():
    """148 SMs x 128 FP32 lanes x max SM clock, lane-ops/s (context beside the measured FFMA rate)."""
    sm_max_mhz = 1965.0
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            sm_max_mhz = float(json.load(f).get("sm_max_mhz", sm_max_mhz))
    except OSError:
        pass
    return N_SM * LANES_PER_SM * sm_max_mhz * 1e6, sm_max_mhz


def kernel_source_sha():
    h = hashlib.sha256()
    for rel in KERNEL_SOURCES:
        with open(os.path.join(ROOT, rel), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def stored_traffic():
    """DRAM bytes per launch from the committed ncu capture -- only if it was taken from the kernel
    source as it stands (profiles/traffic.json carries the hash of the kernel files)."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            t = json.load(f)
    except OSError:
        return None, "profiles/traffic.json missing"
    if t.get("kernel_source_sha") != kernel_source_sha():
        return None, "profiles/traffic.json is stale (kernel source changed since the ncu capture)"
    return t.get("knn_lattice_kernel_dram_bytes_per_launch"), t.get("source")


def stratified_masks(masks, per_dim, seed):
    pc = workloads.popcount(masks)
    rng = np.random.default_rng(seed)
    sel = [rng.choice(np.flatnonzero(pc == d), min(per_dim, int((pc == d).sum())), replace=False)
           for d in np.unique(pc)]
    return masks[np.sort(np.concatenate(sel))]


def oracle_sample(cfg, X, masks, n_queries, seed=0):
    """The T1 oracle on a bounded sample: ~2 masks per dimension x n_queries sampled queries,
    each against all N candidates.  -> (seconds, evals, cores, description)."""
    import oracle
    oracle.build()
    sm = stratified_masks(masks, 2, seed)
    rng = np.random.default_rng(seed + 1)
    q = np.sort(rng.choice(len(X), min(n_queries, len(X)), replace=False))
    t0 = time.perf_counter()
    oracle.knn_selfjoin(X, sm, cfg.k, queries=q)
    dt = time.perf_counter() - t0
    evals = float(len(sm)) * len(q) * len(X)
    what = (f"{len(sm)} subspaces (2 per dimension d=2..15) x {len(q)} sampled queries x all "
            f"{len(X)} candidates, k={cfg.k}, fp64 brute force; subspaces/s = evals/s / N^2")
    return dt, evals, oracle.num_threads(), what


def kdtree_sample(cfg, X, masks, budget_s=15.0, seed=0):
    """A second, library CPU arm beside the oracle (context only): scipy's cKDTree built per subspace and queried
    for all N objects with all host cores -- what a CPU user of the method would run per feature space.  One mask
    per dimension d = 2..15, stopped after `budget_s` seconds; subspaces/s = masks done / time."""
    from scipy.spatial import cKDTree
    sm = stratified_masks(masks, 1, seed)
    t0 = time.perf_counter()
    done, dims = 0, []
    for m in sm:
        cols = [j for j in range(X.shape[1]) if (int(m) >> j) & 1]
        Xs = np.ascontiguousarray(X[:, cols], dtype=np.float64)
        cKDTree(Xs).query(Xs, k=cfg.k + 1, workers=-1)
        done += 1
        dims.append(len(cols))
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    return {"value": done / dt, "unit": UNIT, "kind": "scipy.spatial.cKDTree per subspace, all host cores (library; context only)",
            "sample": f"{done} subspaces, one per dimension (d = {min(dims)}..{max(dims)}), all {len(X)} queries, k={cfg.k}",
            "seconds": dt}


def run_reference(args, rank):
    """--impl reference: the oracle as it stands on the host cores (rank 0 only)."""
    if rank != 0:
        return
    cfg = workloads.get_config(args.config)
    X, masks = cfg.table(), cfg.masks()
    n2 = float(len(X)) ** 2
    for _ in range(args.warmup):
        oracle_sample(cfg, X, masks, 64)
    tot_t, tot_e, cores, what = 0.0, 0.0, 0, ""
    for s in range(args.steps):
        dt, ev, cores, what = oracle_sample(cfg, X, masks, args.ref_queries, seed=s)
        tot_t += dt
        tot_e += ev
    evals_per_s = tot_e / tot_t
    value = evals_per_s / n2
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "evals_per_s": evals_per_s,
        "config": {"workload": workload_name(cfg, len(masks)), "sampled": True},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "each step: " + what},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_name(cfg, n_masks):
    return (f"{cfg.name}: kNNSJ k={cfg.k} over N={cfg.n} x {cfg.n_feat} fp32 (SNAPShot1-shaped, "
            f"seed {cfg.seed}), all {n_masks} subspaces of 2-15 features, scores kth/mean/indeg")


class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                 "-lms", "200", "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            pass
        # nvidia-smi takes 1-2 s to attach to the GPU and host-side CUDA calls stall meanwhile (measured: a
        # one-off 1.8 s in the first timed pass of the LSST-scale leg): wait for its first sample, so that the
        # timed region holds samples, not the start-up
        t0 = time.time()
        while self.p is not None and self.p.poll() is None and time.time() - t0 < 10.0:
            if os.path.getsize(self.f.name) > 0:
                break
            time.sleep(0.05)

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.p.terminate()
        self.p.wait()
        self.f.flush()
        self.f.seek(0)
        rows = [[c.strip() for c in ln.split(",")] for ln in self.f if ln.strip()]
        self.f.close()
        os.unlink(self.f.name)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        sm, reasons, smax, pw = [], set(), None, []
        for r in rows:
            try:
                sm.append(float(r[0]))
                smax = float(r[1])
                pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "power_w_max": max(pw) if pw else None, "samples": len(sm),
                "reasons": sorted(reasons)}


class Dist:
    """torch.distributed plumbing of one run (NCCL for barriers, the max over ranks and the
    in-degree sum; no collective touches the join itself)."""

    def __init__(self, torch, dist, dev, rank, world):
        self.torch, self.dist, self.dev, self.rank, self.world = torch, dist, dev, rank, world

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()

    def max_over_ranks(self, x):
        if self.world == 1:
            return x
        t = self.torch.tensor([x], dtype=self.torch.float64, device=self.dev)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(self, x):
        if self.world == 1:
            return x
        t = self.torch.tensor([x], dtype=self.torch.float64, device=self.dev)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        return float(t.item())


def measured_peak(snaps, local_rank):
    """FFMA / FADD / FADD+FSETP lane-op rates of the in-library probes, with the clocks seen during them."""
    sampler = ClockSampler(local_rank)
    kinds = {"ffma": 0, "fadd": 1, "fadd+fsetp": 2, "ffma_3reg": 3, "ffma2_packed": 4, "fadd2_packed": 5}
    rates = {name: 0.0 for name in kinds}
    for _ in range(3):          # a second of probes so that the 200 ms clock sampler sees them
        for name, kind in kinds.items():
            rates[name] = max(rates[name], snaps.probe_fp32_rate(kind))
    return rates, sampler.stop()


def alu_roofline(kernel, evals, n_batches, N, k_ms, peak_meas, peak_der, sm_max, probes, probe_clocks):
    """bound = plain FP32/ALU issue.  achieved = algorithmic lane-ops / kernel time; peak = the measured
    FFMA lane-op rate.  frac_evals_only drops the per-(pair, batch) term, which depends on the batch size."""
    lane_ops = 2.0 * evals + 30.0 * float(N) * N * n_batches
    achieved = lane_ops / (k_ms * 1e-3)
    return {
        "bound": "alu", "kernel": kernel, "achieved": achieved / 1e12, "peak": peak_meas / 1e12,
        "unit": "TFLOP/s", "frac": achieved / peak_meas,
        "frac_evals_only": 2.0 * evals / (k_ms * 1e-3) / peak_meas,
        "peak_source": "measured: snaps_probe_fp32_rate FFMA lane-ops/s on this GPU during this run (one FFMA = 1 lane-op)",
        "peak_derived": peak_der / 1e12,
        "peak_derived_source": f"{N_SM} SMs x {LANES_PER_SM} FP32 lanes x {sm_max:.0f} MHz",
        "frac_of_fma2_peak": achieved / (2 * peak_meas),
        "probe_lane_ops_per_s": probes, "probe_clocks": probe_clocks,
        "kernel_ms": k_ms, "algorithmic_lane_ops_per_launch": lane_ops,
        "evals_per_s_kernel": evals / (k_ms * 1e-3),
        "note": "effective figure: algorithmic lane-ops (2 per (pair, subspace) evaluation + 30 per pair and batch) / "
                "kernel time.  The kernel reaches the exact result with fewer executed operations (lower-bound filter); "
                "executed-instruction and pipe figures (issue-slot, ALU, FMA utilisation) are in profiles/ (see profiles/README.md)",
    }


def run_lsst(args, cfg, snaps, torch, D, steps, emit=True):
    """LSST-scale config (BASELINE.json configs[3]): N=1,000,000, the 105 two-feature subspaces + the
    full space, k=10, lists and scores streamed to pinned host memory through the grid engine.
    Multi-GPU: query ranges (`sharding.shard_queries`), in-degree rows summed over ranks."""
    from paper_2405_20176_b200.sharding import shard_queries
    X = workloads.make_table(cfg.n, cfg.seed, cols=list(range(cfg.n_feat)), outlier_frac=0.001)
    masks = cfg.masks()
    N, n_masks, k = len(X), len(masks), cfg.k
    q0, q1 = shard_queries(N, D.rank, D.world)
    Xd = torch.from_numpy(X).to(D.dev)
    mpb = 27   # four groups: a group's join overlaps the previous group's copy-out
    out = snaps.knn_selfjoin_streamed(Xd, masks, k, mpb, lists=True, q_range=(q0, q1))
    torch.cuda.synchronize()
    ws = out.pop("_workspace")
    # a second untimed pass: DMA writes into freshly pinned host pages are slow the first TWO times a page is
    # written (1.8 s of host-side stall per pass over these 9.75 GB, then 0.09 s to enqueue a pass)
    snaps.knn_selfjoin_streamed(Xd, masks, k, mpb, lists=True, out=out, workspace=ws, q_range=(q0, q1))
    torch.cuda.synchronize()
    snaps.profile_enable(True)
    D.barrier()
    sampler = ClockSampler(D.dev.index or 0) if D.rank == 0 else None
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kernel_ms = []
    ev0.record()
    for _ in range(steps):
        snaps.knn_selfjoin_streamed(Xd, masks, k, mpb, lists=True, out=out, workspace=ws, q_range=(q0, q1))
        torch.cuda.current_stream().synchronize()
        kernel_ms.append(snaps.profile_last_kernel_ms()[0])
        if D.world > 1:     # the one exchange of query-range sharding: in-degree rows add up
            ind = out["indeg"].to(D.dev, non_blocking=True)
            D.dist.all_reduce(ind)
    ev1.record()
    torch.cuda.synchronize()
    D.barrier()
    clocks = sampler.stop() if sampler else None
    ms = D.max_over_ranks(ev0.elapsed_time(ev1) / steps)
    tot = D.sum_over_ranks(float(out["indeg"][0].sum().item()))
    assert int(tot) == N * k, (tot, N * k)
    if D.rank != 0:
        return None
    evals = float(N) * N * n_masks
    d2h = int(sum(t.numel() * t.element_size() for t in out.values())) * D.world
    line = {
        "metric": "subspaces/sec (kNNSJ N=1,000,000, k=10, 105 pair subspaces + full space, grid engine)",
        "value": n_masks / (ms * 1e-3), "unit": UNIT, "n_gpus": D.world, "steps": steps, "warmup": 2,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": f"{cfg.name}: kNNSJ k={k} over N={N} x 15 (LSST-scale, seed {cfg.seed}), "
                               f"{n_masks} subspaces, lists + scores to pinned host in groups of {mpb} masks",
                   "sharding": "query ranges over ranks; in-degree rows all-reduced" if D.world > 1 else "none"},
        "effective_evals_per_s": evals / (ms * 1e-3),
        "join_kernel_ms": float(np.mean(kernel_ms)),
        "note": "exactly pruned scan (grid index per subspace): effective evals = N^2 x masks / time, not operations performed",
        "e2e": {"value": n_masks / (ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": d2h},
        "clocks": clocks,
        "paper_context": "paper, LSST5M (N=5e6, k_max=256): ~100 s per feature space on 1xA100 (Table 4)"}
    if emit:
        print(json.dumps(line), flush=True)
    return line


def run_range(args, cfg, snaps, torch, D, steps, warmup, peakinfo, emit=True):
    """DSSJ config (BASELINE.json configs[2]): snaps_range_selfjoin over all masks with the stored
    eps_d of the configuration (workloads/config_eps.json)."""
    from paper_2405_20176_b200.sharding import shard_masks
    X = workloads.make_table(cfg.n, cfg.seed, cols=list(range(cfg.n_feat)), outlier_frac=0.01)
    masks_all = cfg.masks()
    eps_all = workloads.config_eps(cfg.name, masks_all)        # stored inputs (oracle/write_config_eps.py)
    if args.masks_limit > 0:                                   # ncu captures only: not a bench value
        masks_all, eps_all = masks_all[:args.masks_limit], eps_all[:args.masks_limit]
    mine = shard_masks(masks_all, D.rank, D.world)
    masks, eps = masks_all[mine], eps_all[mine]
    N, n_masks = len(X), len(masks_all)
    Xd = torch.from_numpy(X).to(D.dev)
    out = snaps.range_selfjoin(Xd, masks, eps)
    ws = out.pop("_workspace")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=D.dev)
    snaps.profile_enable(True)

    def step():
        flush.zero_()
        snaps.range_selfjoin(Xd, masks, eps, out=out, workspace=ws)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    D.barrier()
    sampler = ClockSampler(D.dev.index or 0) if D.rank == 0 else None
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kernel_ms = []
    ev0.record()
    for _ in range(steps):
        step()
        kernel_ms.append(snaps.profile_last_kernel_ms()[0])
    ev1.record()
    torch.cuda.synchronize()
    D.barrier()
    clocks = sampler.stop() if sampler else None
    ms = D.max_over_ranks(ev0.elapsed_time(ev1) / steps)
    if D.rank != 0:
        return None
    evals = float(N) * N * len(masks)            # this rank's share (the kernel time is this rank's)
    n_batches = float(snaps.planned_evals(N, X.shape[1], masks)) / (64.0 * N * N)
    line = {
        **({"partial": f"first {args.masks_limit} masks only (--masks-limit): not a bench value"} if args.masks_limit > 0 else {}),
        "metric": "subspaces/sec (DSSJ N=31,693, eps_d for ~50 neighbours)", "value": n_masks / (ms * 1e-3),
        "unit": UNIT, "n_gpus": D.world, "steps": steps, "warmup": warmup, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{cfg.name}: DSSJ over N={N} x 15 (seed {cfg.seed}), all {n_masks} subspaces, counts + sums + means",
                   "l2": "256 MB flush fill before every step"},
        "evals_per_s": float(N) * N * n_masks / (ms * 1e-3),
        "mean_neighbours": float(out["count"].float().mean().item()),
        "roofline": alu_roofline("range_lattice_kernel", evals, n_batches, N, float(np.mean(kernel_ms)), *peakinfo),
        "gpu_launches": 4 * steps, "clocks": clocks}
    if emit:
        print(json.dumps(line), flush=True)
    return line


def run_select_k(args, cfg, snaps, torch, D, n_masks=None, steps=None, warmup=None, emit=True):
    """The kNN parameter selection of PAPER.md:181-189, 258-260 at the paper's SNAPShot1 operating point: one join at
    k_max = 4096 gives every smaller k's lists as prefixes; snaps_knn_select_k then forms the scores at
    every k_j of the grid, ranks them, and takes Eq. 2 against the smallest and largest k and Eq. 3 -- for both kNN
    metrics.  The paper's k grid is "unevenly sampled" and not printed (reading A17): powers of two 2 ... 4096 here."""
    X = workloads.make_table(cfg.n, cfg.seed, cols=list(range(cfg.n_feat)), outlier_frac=0.01)
    N = len(X)
    masks_all = cfg.masks()
    n_steps, n_warm = steps or args.steps, warmup if warmup is not None else max(1, args.warmup)
    masks = masks_all[np.linspace(0, len(masks_all) - 1, n_masks or args.select_k).astype(np.int64)]
    k_max, n_top = 4096, int(round(0.01 * N))
    k_grid = np.array([2, 4, 8, 16, 32, 64, 128, 256, 512, 1024, 2048, 3072, 4096], dtype=np.int32)
    Xd = torch.from_numpy(X).to(D.dev)
    chunk = 8
    first = snaps.knn_selfjoin(Xd, masks[:chunk], k_max, engine="grid")
    ws = first.pop("_workspace")
    snaps.profile_enable(True)
    join_ms = []

    def step():
        for m0 in range(0, len(masks), chunk):
            mm = masks[m0:m0 + chunk]
            if len(mm) == chunk:
                j = snaps.knn_selfjoin(Xd, mm, k_max, engine="grid", out=first, workspace=ws)
            else:
                j = snaps.knn_selfjoin(Xd, mm, k_max, engine="grid")
            join_ms.append(snaps.profile_last_kernel_ms()[0])
            sel = snaps.knn_select_k(j["idx"], j["dist"], k_grid, n_top)
        return sel

    for _ in range(n_warm):
        step()
    torch.cuda.synchronize()
    join_ms.clear()
    sampler = ClockSampler(D.dev.index or 0)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(n_steps):
        sel = step()
    ev1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1) / n_steps
    line = {
        "metric": "feature spaces/sec (kNN parameter selection: join at k_max = 4096 + scores at 13 k + ranks + Eq. 2 + Eq. 3)",
        "value": len(masks) / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": n_steps, "warmup": n_warm,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{cfg.name}: N={N} x 15 (seed {cfg.seed}), {len(masks)} subspaces spread over the 32,752, "
                               f"k_max={k_max}, k grid {k_grid.tolist()}, top {n_top}"},
        "ms_per_subspace": ms / len(masks), "join_ms_per_subspace": float(np.sum(join_ms)) / n_steps / len(masks),
        "seconds_for_all_32752": ms / len(masks) * 32752 / 1e3,
        "selected_grid_index_histogram_last_chunk": np.bincount(sel["j_mean"].cpu().numpy(), minlength=len(k_grid)).tolist(),
        "clocks": clocks,
        "paper_context": "paper: kNNSJ more expensive than DSSJ (PAPER.md:398); absolute kNNSJ time on SNAPShot1 not in the "
                         "text (Fig. 10 is an image)"}
    if emit:
        print(json.dumps(line), flush=True)
    return line


def run_select_eps(args, cfg, snaps, torch, D, n_masks=None, steps=None, warmup=None, emit=True):
    """The DSSJ parameter selection of PAPER.md:181-189, 229-239 in one call per chunk of masks
    (snaps_range_select_eps: eps_min / eps_max search -> |G| radii -> one join at eps_max -> ranks -> Eq. 2 -> Eq. 3)
    at the paper's operating point on SNAPShot1: s_min = 0.001 |D|, s_max = 0.15 |D|, |G| = 22 (Fig. 2,
    reading A22), top 1 %.  The paper's figure for this workload over all 32,752 feature spaces,
    whole pipeline on 1 x A100 with o = 8: 2.64 h -- context, other hardware."""
    X = workloads.make_table(cfg.n, cfg.seed, cols=list(range(cfg.n_feat)), outlier_frac=0.01)
    N = len(X)
    groups = {}
    for m in cfg.masks():
        groups.setdefault(int(m) >> 6, []).append(m)
    keys = sorted(groups)
    n_steps, n_warm = steps or args.steps, warmup if warmup is not None else max(1, args.warmup)
    n_b = max(1, (n_masks or args.select_eps) // 64)
    masks = np.array([m for kk in keys[::max(1, len(keys) // n_b)][:n_b] for m in groups[kk]], dtype=np.uint16)
    rng = np.random.default_rng(cfg.seed)
    q = np.sort(rng.choice(N, 1000, replace=False)).astype(np.int32)
    c = np.arange(N, dtype=np.int32)
    G, n_top, s_min, s_max = 22, int(round(0.01 * N)), 0.001 * N, 0.15 * N
    Xd = torch.from_numpy(X).to(D.dev)
    chunk = 512

    def step():
        for m0 in range(0, len(masks), chunk):
            out = snaps.range_select_eps(Xd, masks[m0:m0 + chunk], q, c, s_min, s_max, G, n_top, 4096, engine="lattice")
        return out

    for _ in range(n_warm):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(D.dev.index or 0)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(n_steps):
        out = step()
    ev1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1) / n_steps
    line = {
        "metric": "feature spaces/sec (DSSJ parameter selection: eps search + 22-radius join at s_max + ranks + Eq. 2 + Eq. 3)",
        "value": len(masks) / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": n_steps, "warmup": n_warm,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{cfg.name}: N={N} x 15 (seed {cfg.seed}), {len(masks)} subspaces = {n_b} whole sub-lattice batches "
                               f"spread over the 32,752, s_min={s_min:.0f}, s_max={s_max:.0f} neighbours, |G|={G}, top {n_top}"},
        "ms_per_subspace": ms / len(masks), "seconds_for_all_32752": ms / len(masks) * 32752 / 1e3,
        "selected_grid_index_histogram_last_chunk": np.bincount(out["j_count"].cpu().numpy(), minlength=G).tolist(),
        "clocks": clocks,
        "paper_context": "paper: DSSJ over all 32,752 feature spaces incl. eps^select and both rankings, 2.64 h on 1xA100 "
                         "(o=8), whole pipeline with CPU post-processing and file output (PAPER.md:394)"}
    if emit:
        print(json.dumps(line), flush=True)
    return line


def run_c5(args, cfg, snaps, torch, D):
    """Config 5 (BASELINE.json configs[4]): N=5,000,000 x 15, 256 subspace masks sampled from the 32,752,
    kNNSJ k=16 plus DSSJ (eps_d for ~100 neighbours), outputs through the recycling sink (two pinned host
    buffers; the consumer checksums each group and the buffer is reused) -- the lists (164 GB) never
    exist anywhere at once.  One pass each (minutes); --c5-n reduces N for quick runs."""
    from paper_2405_20176_b200.sharding import shard_queries
    n = args.c5_n or cfg.n
    X = workloads.make_table(n, cfg.seed, cols=list(range(cfg.n_feat)), outlier_frac=0.001)
    masks = cfg.masks()
    if args.c5_masks:
        masks = masks[:args.c5_masks]
    N, n_masks, k = len(X), len(masks), cfg.k
    q0, q1 = shard_queries(N, D.rank, D.world)
    Xd = torch.from_numpy(X).to(D.dev)
    mpb = 4
    acc = {"kth": 0.0, "indeg": 0, "groups": 0, "idx_xor": 0, "count": 0, "bytes": 0}

    def consume_knn(m0, m1, arrays):
        acc["groups"] += 1
        acc["kth"] += float(arrays["kth"].sum(dtype=np.float64))
        acc["indeg"] += int(arrays["indeg"].sum(dtype=np.int64))
        acc["idx_xor"] ^= int(np.bitwise_xor.reduce(arrays["idx"][:, ::997].ravel()))
        acc["bytes"] += sum(a.nbytes for a in arrays.values())

    def consume_range(m0, m1, arrays):
        acc["count"] += int(arrays["count"].sum(dtype=np.int64))
        acc["bytes"] += sum(a.nbytes for a in arrays.values())

    # radii for ~100 neighbours: the library's own sampled-histogram search (NEXT-2) on the device
    eps = snaps.eps_for_selectivity(Xd, masks, cfg.target_neighbours, seed=cfg.seed)
    snaps.profile_enable(True)
    D.barrier()
    sampler = ClockSampler(D.dev.index or 0) if D.rank == 0 else None
    t = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    t[0].record()
    ws = snaps.knn_selfjoin_sink(Xd, masks, k, mpb, consume_knn, want=("idx", "dist", "kth", "mean", "indeg"),
                                 q_range=(q0, q1))
    knn_kernel_ms = snaps.profile_last_kernel_ms()[0]
    t[1].record()
    snaps.range_selfjoin_sink(Xd, masks, eps, mpb, consume_range, q_range=(q0, q1), workspace=ws)
    rng_kernel_ms = snaps.profile_last_kernel_ms()[0]
    t[2].record()
    torch.cuda.synchronize()
    D.barrier()
    clocks = sampler.stop() if sampler else None
    knn_ms = D.max_over_ranks(t[0].elapsed_time(t[1]))
    rng_ms = D.max_over_ranks(t[1].elapsed_time(t[2]))
    indeg = D.sum_over_ranks(float(acc["indeg"]))
    cnt = D.sum_over_ranks(float(acc["count"]))
    assert int(indeg) == N * k * n_masks, (indeg, N * k * n_masks)       # PAPER.md:136 over every mask
    if D.rank != 0:
        return
    evals = float(N) * N * n_masks
    print(json.dumps({
        "metric": "subspaces/sec (kNNSJ k=16 + DSSJ ~100 neighbours, N=5,000,000, 256 sampled subspaces, grid engine, sink)",
        "value": n_masks / ((knn_ms + rng_ms) * 1e-3), "unit": UNIT, "n_gpus": D.world, "steps": 1, "warmup": 0,
        "ms_per_step": knn_ms + rng_ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{cfg.name}: N={N} x 15 (seed {cfg.seed}), {n_masks} masks sampled from the 32,752 (seed 4), "
                               f"kNNSJ k={k} (lists + scores) then DSSJ (counts, sums, means), groups of {mpb} masks "
                               "through two recycled pinned host buffers"},
        "knn": {"ms": knn_ms, "subspaces_per_s": n_masks / (knn_ms * 1e-3), "effective_evals_per_s": evals / (knn_ms * 1e-3),
                "join_kernel_ms": knn_kernel_ms, "s_per_subspace": knn_ms * 1e-3 / n_masks},
        "dssj": {"ms": rng_ms, "subspaces_per_s": n_masks / (rng_ms * 1e-3), "effective_evals_per_s": evals / (rng_ms * 1e-3),
                 "join_kernel_ms": rng_kernel_ms, "mean_neighbours": cnt / (float(N) * n_masks)},
        "e2e": {"value": n_masks / ((knn_ms + rng_ms) * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 0,
                "d2h_bytes_per_step": int(acc["bytes"]) * D.world},
        "sink": {"groups": acc["groups"], "kth_checksum": acc["kth"], "idx_xor": acc["idx_xor"]},
        "clocks": clocks,
        "paper_context": "paper, LSST5M on 1xA100 (k_max=256, s_max=256): kNNSJ ~100 s, DSSJ ~24 s per feature space (Table 4)",
    }), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="snaps", choices=["snaps", "reference"])
    ap.add_argument("--config", default="c2_snapshot1_knn")
    ap.add_argument("--scaling", default="strong", choices=["strong", "weak"],
                    help="N > 1: strong = one catalogue, masks dealt to ranks; weak = one catalogue per rank")
    ap.add_argument("--dealing", default="static", choices=["static", "dynamic"],
                    help="strong scaling of config 2: static = batches dealt round-robin up front; dynamic = a shared "
                         "counter hands out groups of 8 batches, the least loaded rank takes the next (PAPER.md:323)")
    ap.add_argument("--ref-queries", type=int, default=1024,
                    help="sampled queries per step of --impl reference")
    ap.add_argument("--cpu-queries", type=int, default=4096,
                    help="sampled queries of the cpu_baseline leg (0 = skip)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-lsst", action="store_true", help="skip the LSST-scale leg (config 4) of the default run")
    ap.add_argument("--no-dssj", action="store_true", help="skip the DSSJ leg (config 3) of the default run")
    ap.add_argument("--no-select", action="store_true", help="skip the parameter-selection legs of the default run")
    ap.add_argument("--masks-limit", type=int, default=0,
                    help="headline step on the first M masks only, for `ncu --set full` captures (ncu replays a launch "
                         "~40 times and saves / restores its 12.5 GB of outputs around each replay); the line is marked "
                         "`partial` and is NOT a bench value")
    ap.add_argument("--select-eps", type=int, default=0, metavar="M",
                    help="with --config c3_snapshot1_dssj: time the DSSJ parameter selection (snaps_range_select_eps) at the "
                         "paper's operating point on M masks (whole sub-lattice batches spread over the mask list) instead of the join")
    ap.add_argument("--select-k", type=int, default=0, metavar="M",
                    help="with the default config: time the kNN parameter selection at the paper's operating point (join at "
                         "k_max = 4096, then snaps_knn_select_k over a 13-point k grid) on M masks spread over the mask list")
    ap.add_argument("--c5-n", type=int, default=0, help="config 5 with a reduced N (quick runs)")
    ap.add_argument("--c5-masks", type=int, default=0, help="config 5 on its first M masks only (quick runs)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    import paper_2405_20176_b200 as snaps
    from paper_2405_20176_b200.sharding import shard_masks

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback exists)"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("NCCL_DEBUG", "INFO")          # the communicator log shows the ranks
        dist.init_process_group("nccl", device_id=dev)
    snaps.lib()
    D = Dist(torch, dist, dev, rank, world)

    cfg = workloads.get_config(args.config)
    probes, probe_clocks = measured_peak(snaps, local_rank)
    peak_der, sm_max = derived_peak()
    peakinfo = (probes["ffma"], peak_der, sm_max, probes, probe_clocks)
    try:
        if cfg.name == "c5_lsst_oversub":
            run_c5(args, cfg, snaps, torch, D)
            return
        if cfg.join == "knn" and cfg.n >= 100000:
            run_lsst(args, cfg, snaps, torch, D, max(1, args.steps))
            return
        if cfg.join == "knn" and args.select_k > 0:
            run_select_k(args, cfg, snaps, torch, D)
            return
        if cfg.join == "range" and args.select_eps > 0:
            run_select_eps(args, cfg, snaps, torch, D)
            return
        if cfg.join == "range":
            run_range(args, cfg, snaps, torch, D, args.steps, args.warmup, peakinfo)
            return
        run_headline(args, cfg, snaps, torch, D, shard_masks, peakinfo)
    finally:
        if world > 1:
            dist.destroy_process_group()


def run_headline(args, cfg, snaps, torch, D, shard_masks, peakinfo):
    rank, world, dev = D.rank, D.world, D.dev
    weak = world > 1 and args.scaling == "weak"
    X = workloads.make_table(cfg.n, cfg.seed + (rank if weak else 0), cols=list(range(cfg.n_feat)), outlier_frac=0.01)
    masks_all = cfg.masks()
    if args.masks_limit > 0:
        masks_all = masks_all[:args.masks_limit]
    dynamic = args.dealing == "dynamic" and not weak
    mine = np.arange(len(masks_all)) if (world == 1 or weak or dynamic) else shard_masks(masks_all, rank, world)
    masks = masks_all[mine]
    N, n_feat, k, n_masks = len(X), X.shape[1], cfg.k, len(masks)
    job_masks = len(masks_all) * (world if weak else 1)       # subspaces the whole job finishes per step
    evals = float(N) * N * n_masks                            # this rank's (pair, subspace) evaluations
    planned = float(snaps.planned_evals(N, n_feat, masks))

    Xd = torch.from_numpy(X).to(dev)
    ws = torch.empty(snaps.workspace_bytes(N, n_feat, n_masks, k), dtype=torch.uint8, device=dev)
    out = {"kth": torch.empty((n_masks, N), dtype=torch.float32, device=dev),
           "mean": torch.empty((n_masks, N), dtype=torch.float32, device=dev),
           "indeg": torch.empty((n_masks, N), dtype=torch.int32, device=dev)}
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2
    snaps.profile_enable(True)

    step_no = [0]
    if dynamic:
        # the least loaded GPU takes the next unit.  Units = groups of 8 sub-lattice batches (512
        # masks); a counter in the job's store hands them out; every rank keeps what it computed in its own rows.
        from paper_2405_20176_b200.sharding import DynamicDealer, mask_groups
        groups = mask_groups(masks_all, 8)
        store = (D.dist.distributed_c10d._get_default_store() if world > 1 else D.dist.HashStore())

    def step():
        """-> (join-kernel ms, join launches, masks this rank processed)"""
        flush.zero_()
        if not dynamic:
            snaps.knn_selfjoin(Xd, masks, k, lists=False, out=out, workspace=ws)
            ms, n = snaps.profile_last_kernel_ms()     # waits for this step's join kernel
            return ms, n + 3, n_masks                  # + the two staging kernels + the L2 flush fill
        step_no[0] += 1
        ms_tot, n_tot, row = 0.0, 1, 0
        for u in DynamicDealer(store, len(groups), name=f"knn_step_{step_no[0]}"):
            g = groups[u]
            sub = {name: t[row:row + len(g)] for name, t in out.items()}
            snaps.knn_selfjoin(Xd, masks_all[g], k, lists=False, out=sub, workspace=ws)
            ms, n = snaps.profile_last_kernel_ms()
            ms_tot, n_tot, row = ms_tot + ms, n_tot + n + 2, row + len(g)
        return ms_tot, n_tot, row

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    D.barrier()
    sampler = ClockSampler(dev.index or 0) if rank == 0 else None
    kernel_ms, launches, done = [], 0, []
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(args.steps):
        ms, n, nm = step()
        kernel_ms.append(ms)
        launches += n
        done.append(nm)
    ev1.record()
    torch.cuda.synchronize()
    D.barrier()
    clocks = sampler.stop() if sampler else None
    ms_per_step = D.max_over_ranks(ev0.elapsed_time(ev1) / args.steps)
    value = job_masks / (ms_per_step * 1e-3)
    evals_per_s = float(N) * N * job_masks / (ms_per_step * 1e-3)

    # sanity on the last step's result: every mask's in-degree row sums to N*k
    if dynamic:
        tot = D.sum_over_ranks(float(done[-1]))
        assert int(tot) == len(masks_all), f"dynamic dealing covered {tot} of {len(masks_all)} masks"
        evals = float(N) * N * float(np.mean(done))               # what this rank processed per step
        planned = evals * float(snaps.planned_evals(N, n_feat, masks_all)) / (float(N) * N * len(masks_all))
    chk = int(out["indeg"][max(0, min(n_masks, done[-1]) // 2)].sum().item()) if done[-1] > 0 else N * k
    assert chk == N * k, f"in-degree sum {chk} != N*k = {N * k}"

    # ---- roofline of the dominant kernel (knn_lattice_kernel): ALU/FP32-issue bound
    k_ms = float(np.mean(kernel_ms))
    n_batches = planned / (64.0 * N * N)
    roofline = alu_roofline("knn_lattice_kernel", evals, n_batches, N, k_ms, *peakinfo)
    roofline["traffic"], roofline["traffic_source"] = stored_traffic()
    roofline["kernel_share_of_step"] = k_ms / ms_per_step
    roofline["planned_lattice_slots_over_masks"] = planned / evals

    # ---- end to end: ONE C call with host buffers (pinned X in, pinned scores out)
    e2e = None
    if not args.no_e2e:
        import psutil
        score_bytes = 3 * 4 * n_masks * N
        if psutil.virtual_memory().available > 3 * score_bytes:
            del out
            torch.cuda.empty_cache()
            Xh = torch.from_numpy(X).pin_memory()
            mpb = 4096           # 8 groups: a group's join overlaps the previous group's copy-out
            hws = torch.empty(snaps.workspace_bytes(N, n_feat, n_masks, k, x_on_host=True) +
                              snaps.stream_ring_bytes(N, N, k, mpb), dtype=torch.uint8, device=dev)
            hout = {"kth": torch.empty((n_masks, N), dtype=torch.float32, pin_memory=True),
                    "mean": torch.empty((n_masks, N), dtype=torch.float32, pin_memory=True),
                    "indeg": torch.empty((n_masks, N), dtype=torch.int32, pin_memory=True)}

            def host_step():
                snaps.knn_selfjoin_host(Xh, masks, k, mpb, lists=False, out=hout, workspace=hws)
                torch.cuda.current_stream().synchronize()
                return float(hout["kth"][-1, -1])          # the host reads the result

            # two untimed passes: DMA writes into freshly pinned host pages are slow the first two times a page is
            # written (measured on the LSST-scale leg: 1.8 s per 9.75 GB, twice, then never again)
            host_step()
            host_step()
            D.barrier()
            t0 = time.perf_counter()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record()
            n_e2e = max(1, min(args.steps, 3))
            for _ in range(n_e2e):
                host_step()
            g1.record()
            torch.cuda.synchronize()
            wall = (time.perf_counter() - t0) / n_e2e
            e_ms = D.max_over_ranks(max(g0.elapsed_time(g1) / n_e2e, wall * 1e3))
            assert int(hout["indeg"][n_masks // 2].sum().item()) == N * k
            e2e = {"value": job_masks / (e_ms * 1e-3), "unit": UNIT,
                   "h2d_bytes_per_step": int(X.nbytes + masks.nbytes) * world,
                   "d2h_bytes_per_step": int(score_bytes) * world, "ms_per_step": e_ms, "steps": n_e2e, "warmup": 2,
                   "api": "snaps_knn_selfjoin_streamed with SNAPS_FLAG_X_ON_HOST: one C call, pinned host table in, "
                          "pinned host scores out"}
            del hout, hws, Xh
        else:
            e2e = {"value": None, "unit": UNIT, "skipped": "host RAM too small for pinned scores"}

    cpu = None
    if rank == 0 and world == 1 and args.cpu_queries > 0:
        dt, ev, cores, what = oracle_sample(cfg, X, masks, args.cpu_queries)
        cpu = {"value": ev / dt / (float(N) * N), "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": what, "evals_per_s": ev / dt, "seconds": dt}
        try:
            cpu["library_arm"] = kdtree_sample(cfg, X, masks)
        except Exception as e:                                   # scipy missing or too slow: the oracle figure stands
            cpu["library_arm"] = {"error": repr(e)[:120]}

    # ---- the other configs, side by side (north star): DSSJ (config 3), LSST scale (config 4)
    dssj = lsst = None
    default_run = world == 1 and args.config == "c2_snapshot1_knn" and args.masks_limit == 0
    Xd = ws = out = None
    torch.cuda.empty_cache()
    if default_run and not args.no_dssj:
        try:
            full = run_range(args, workloads.get_config("c3_snapshot1_dssj"), snaps, torch, D, 3, 1, peakinfo, emit=False)
            dssj = {k_: full[k_] for k_ in ("metric", "value", "unit", "steps", "ms_per_step", "evals_per_s",
                                            "mean_neighbours", "roofline", "clocks")}
            dssj["workload"] = full["config"]["workload"]
        except Exception as e:                                   # the headline line must survive this leg
            dssj = {"error": repr(e)[:200]}
        torch.cuda.empty_cache()
    if default_run and not args.no_lsst:
        try:
            full = run_lsst(args, workloads.get_config("c4_lsst_pairs"), snaps, torch, D, 3, emit=False)
            lsst = {k_: full[k_] for k_ in ("metric", "value", "unit", "steps", "ms_per_step", "effective_evals_per_s",
                                            "join_kernel_ms", "note", "clocks")}
            lsst["workload"] = full["config"]["workload"]
            lsst["d2h_bytes_per_step"] = full["e2e"]["d2h_bytes_per_step"]
        except Exception as e:
            lsst = {"error": repr(e)[:200]}

    select = None
    if default_run and not args.no_select:
        # the paper's own operating points, a few seconds each: parameter selection for DSSJ at
        # s_max = 0.15 N over 22 radii, and for kNN at k_max = 4096
        select = {}
        for name, fn, cfgname, nm in (("eps", run_select_eps, "c3_snapshot1_dssj", 512), ("k", run_select_k, "c2_snapshot1_knn", 16)):
            try:
                torch.cuda.empty_cache()
                full = fn(args, workloads.get_config(cfgname), snaps, torch, D, n_masks=nm, steps=2, warmup=1, emit=False)
                select[name] = {k_: full[k_] for k_ in ("metric", "value", "unit", "steps", "ms_per_step", "ms_per_subspace",
                                                        "seconds_for_all_32752", "clocks")}
                select[name]["workload"] = full["config"]["workload"]
            except Exception as e:
                select[name] = {"error": repr(e)[:200]}

    if rank == 0:
        line = {
            **({"partial": f"first {args.masks_limit} masks only (--masks-limit): not a bench value"} if args.masks_limit > 0 else {}),
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak" if weak else "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(cfg, len(masks_all)),
                       "l2": "256 MB flush fill before every step; each step also writes 12.5 GB of scores",
                       "outputs": "scores only (lists of this config are 83 GB)",
                       "sharding": ("one catalogue per rank" if weak else
                                    "one catalogue; groups of 8 batches handed out by a shared counter (least loaded rank next), no collective"
                                    if dynamic else
                                    "one catalogue; masks dealt to ranks by sub-lattice batch, no collective") if (world > 1 or dynamic) else "none"},
            "evals_per_s": evals_per_s, "fp32_peak_frac": roofline["frac"],
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches,
            "dssj": dssj, "lsst_scale": lsst, "parameter_selection": select,
            "clocks": clocks,
            "paper_context": "paper: DSSJ all 32,752 spaces 2.64 h on 1xA100 (o=8) incl. CPU "
                             "post-processing; LSST5M kNNSJ ~100 s/feature space (PAPER.md:394, Table 4)",
        }
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
