"""ctypes binding for libsnaps.so -- same names as include/snaps.h, marshalling only."""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

EXPORTED_SYMBOLS = [
    "snaps_last_error", "snaps_version", "snaps_workspace_bytes", "snaps_planned_evals",
    "snaps_knn_selfjoin", "snaps_range_selfjoin", "snaps_outlier_scores",
    "snaps_stream_ring_bytes", "snaps_knn_selfjoin_streamed", "snaps_probe_fp32_rate",
    "snaps_profile_enable", "snaps_profile_last_kernel_ms",
    "snaps_rank_workspace_bytes", "snaps_rank_scores", "snaps_topn_overlap", "snaps_select_parameter",
    "snaps_knn_scores_at_k", "snaps_range_grid_workspace_bytes", "snaps_range_selfjoin_grid",
    "snaps_select_k_workspace_bytes", "snaps_knn_select_k",
    "snaps_dist_hist_workspace_bytes", "snaps_sample_distance_histogram", "snaps_eps_from_histogram",
]

_lib = None


class SnapsError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"snaps status {status}: {message}")
        self.status = status


def lib_path() -> str:
    return _build.LIB


def lib():
    """Load libsnaps.so (building it in-tree if missing).  Fails loudly if it cannot."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        i64, i32, vp, sz = ctypes.c_int64, ctypes.c_int, ctypes.c_void_p, ctypes.c_size_t
        L.snaps_last_error.restype = ctypes.c_char_p
        L.snaps_version.restype = ctypes.c_char_p
        L.snaps_workspace_bytes.restype = sz
        L.snaps_workspace_bytes.argtypes = [i64, i32, i32, i32]
        L.snaps_planned_evals.restype = i64
        L.snaps_planned_evals.argtypes = [i64, i32, vp, i32]
        L.snaps_knn_selfjoin.restype = i32
        L.snaps_knn_selfjoin.argtypes = [vp, i64, i32, i64, vp, i32, i32, vp, vp, vp, vp, vp, vp, sz, vp]
        L.snaps_range_selfjoin.restype = i32
        L.snaps_range_selfjoin.argtypes = [vp, i64, i32, i64, vp, i32, vp, vp, vp, vp, vp, sz, vp]
        L.snaps_outlier_scores.restype = i32
        L.snaps_outlier_scores.argtypes = [i64, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.snaps_stream_ring_bytes.restype = sz
        L.snaps_stream_ring_bytes.argtypes = [i64, i32, i32]
        L.snaps_knn_selfjoin_streamed.restype = i32
        L.snaps_knn_selfjoin_streamed.argtypes = [vp, i64, i32, i64, vp, i32, i32, i32,
                                                  vp, vp, vp, vp, vp, vp, sz, vp]
        L.snaps_probe_fp32_rate.restype = i32
        L.snaps_probe_fp32_rate.argtypes = [i32, ctypes.POINTER(ctypes.c_double), vp]
        L.snaps_profile_enable.restype = i32
        L.snaps_profile_enable.argtypes = [i32]
        L.snaps_profile_last_kernel_ms.restype = i32
        L.snaps_profile_last_kernel_ms.argtypes = [ctypes.POINTER(ctypes.c_float),
                                                   ctypes.POINTER(ctypes.c_int)]
        L.snaps_rank_workspace_bytes.restype = sz
        L.snaps_rank_workspace_bytes.argtypes = [i64, i32]
        L.snaps_rank_scores.restype = i32
        L.snaps_rank_scores.argtypes = [i32, vp, vp, i64, i32, vp, vp, vp, sz, vp]
        L.snaps_topn_overlap.restype = i32
        L.snaps_topn_overlap.argtypes = [vp, vp, i64, i32, i32, vp, vp]
        L.snaps_select_parameter.restype = i32
        L.snaps_select_parameter.argtypes = [vp, vp, i32, i32, i32, vp, vp]
        L.snaps_range_grid_workspace_bytes.restype = sz
        L.snaps_range_grid_workspace_bytes.argtypes = [i64, i32, i32, i32]
        L.snaps_range_selfjoin_grid.restype = i32
        L.snaps_range_selfjoin_grid.argtypes = [vp, i64, i32, i64, vp, i32, vp, i32, vp, vp, vp, vp, sz, vp]
        L.snaps_dist_hist_workspace_bytes.restype = sz
        L.snaps_dist_hist_workspace_bytes.argtypes = [i32, i32, i32]
        L.snaps_sample_distance_histogram.restype = i32
        L.snaps_sample_distance_histogram.argtypes = [vp, i64, i32, i64, vp, i32, vp, i32, vp, i32, vp, i32, vp, vp, sz, vp]
        L.snaps_eps_from_histogram.restype = i32
        L.snaps_eps_from_histogram.argtypes = [vp, i32, i32, vp, i64, i64, ctypes.c_double, vp]
        L.snaps_select_k_workspace_bytes.restype = sz
        L.snaps_select_k_workspace_bytes.argtypes = [i64, i32]
        L.snaps_knn_select_k.restype = i32
        L.snaps_knn_select_k.argtypes = [i64, i32, i32, vp, vp, vp, i32, i32, vp, vp, vp, vp, sz, vp]
        L.snaps_knn_scores_at_k.restype = i32
        L.snaps_knn_scores_at_k.argtypes = [i64, i32, i32, i32, vp, vp, vp, vp, vp, vp]
        _lib = L
    return _lib


def _check(status: int):
    if status != 0:
        raise SnapsError(status, lib().snaps_last_error().decode())


def version() -> str:
    return lib().snaps_version().decode()


def _masks(masks) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(masks, dtype=np.uint16).ravel())


def _dptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def workspace_bytes(N: int, n_feat: int, n_masks: int, k: int) -> int:
    return int(lib().snaps_workspace_bytes(N, n_feat, n_masks, k))


def stream_ring_bytes(N: int, k: int, masks_per_batch: int) -> int:
    return int(lib().snaps_stream_ring_bytes(N, k, masks_per_batch))


def planned_evals(N: int, n_feat: int, masks) -> int:
    m = _masks(masks)
    return int(lib().snaps_planned_evals(N, n_feat, m.ctypes.data_as(ctypes.c_void_p), len(m)))


def _workspace(X, n_masks, k, extra=0):
    import torch
    nbytes = workspace_bytes(X.shape[0], X.shape[1], n_masks, k) + extra
    if nbytes == 0:
        raise SnapsError(1, "invalid sizes for workspace")
    return torch.empty(nbytes, dtype=torch.uint8, device=X.device)


def knn_selfjoin(X, masks, k, *, lists=True, scores=True, out=None, workspace=None, stream=None):
    """snaps_knn_selfjoin on a CUDA fp32 tensor X [N, n_feat].

    Returns a dict with idx/dist [n_masks, N, k] (if lists) and kth/mean/indeg [n_masks, N]
    (if scores), all torch CUDA tensors.  `out` may supply preallocated tensors by those names."""
    import torch
    assert X.is_cuda and X.dtype == torch.float32 and X.dim() == 2 and X.stride(1) == 1
    m = _masks(masks)
    N, n_feat = X.shape
    out = dict(out or {})
    dev = X.device
    if lists:
        out.setdefault("idx", torch.empty((len(m), N, k), dtype=torch.int32, device=dev))
        out.setdefault("dist", torch.empty((len(m), N, k), dtype=torch.float32, device=dev))
    if scores:
        out.setdefault("kth", torch.empty((len(m), N), dtype=torch.float32, device=dev))
        out.setdefault("mean", torch.empty((len(m), N), dtype=torch.float32, device=dev))
        out.setdefault("indeg", torch.empty((len(m), N), dtype=torch.int32, device=dev))
    ws = workspace if workspace is not None else _workspace(X, len(m), k)
    _check(lib().snaps_knn_selfjoin(
        _dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m), k,
        _dptr(out.get("idx")), _dptr(out.get("dist")), _dptr(out.get("kth")),
        _dptr(out.get("mean")), _dptr(out.get("indeg")), _dptr(ws), ws.numel(), _stream(stream)))
    out["_workspace"] = ws
    return out


def range_selfjoin(X, masks, eps, *, sums=True, out=None, workspace=None, stream=None):
    """snaps_range_selfjoin: returns dict count [n_masks, N] (int32 view of uint32) and, if
    sums, sumdist / mean."""
    import torch
    assert X.is_cuda and X.dtype == torch.float32 and X.dim() == 2 and X.stride(1) == 1
    m = _masks(masks)
    e = np.ascontiguousarray(np.asarray(eps, dtype=np.float32).ravel())
    assert len(e) == len(m)
    N, n_feat = X.shape
    out = dict(out or {})
    dev = X.device
    out.setdefault("count", torch.empty((len(m), N), dtype=torch.int32, device=dev))
    if sums:
        out.setdefault("sumdist", torch.empty((len(m), N), dtype=torch.float32, device=dev))
        out.setdefault("mean", torch.empty((len(m), N), dtype=torch.float32, device=dev))
    ws = workspace if workspace is not None else _workspace(X, len(m), 0)
    _check(lib().snaps_range_selfjoin(
        _dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m),
        e.ctypes.data_as(ctypes.c_void_p), _dptr(out["count"]), _dptr(out.get("sumdist")),
        _dptr(out.get("mean")), _dptr(ws), ws.numel(), _stream(stream)))
    out["_workspace"] = ws
    return out


def outlier_scores(N, n_masks, k, *, knn_idx=None, knn_dist=None, eps_count=None, eps_sumdist=None,
                   stream=None):
    """snaps_outlier_scores from join outputs on the device."""
    import torch
    ref = next(t for t in (knn_idx, knn_dist, eps_count, eps_sumdist) if t is not None)
    dev = ref.device
    out = {}
    if knn_dist is not None:
        out["kth"] = torch.empty((n_masks, N), dtype=torch.float32, device=dev)
        out["mean"] = torch.empty((n_masks, N), dtype=torch.float32, device=dev)
    if knn_idx is not None:
        out["indeg"] = torch.empty((n_masks, N), dtype=torch.int32, device=dev)
    if eps_count is not None and eps_sumdist is not None:
        out["eps_mean"] = torch.empty((n_masks, N), dtype=torch.float32, device=dev)
    _check(lib().snaps_outlier_scores(
        N, n_masks, k, _dptr(knn_idx), _dptr(knn_dist), _dptr(eps_count), _dptr(eps_sumdist),
        _dptr(out.get("kth")), _dptr(out.get("mean")), _dptr(out.get("indeg")),
        _dptr(out.get("eps_mean")), _stream(stream)))
    return out


def knn_selfjoin_streamed(X, masks, k, masks_per_batch, *, lists=True, scores=True, out=None,
                          workspace=None, stream=None):
    """snaps_knn_selfjoin_streamed: outputs land in PINNED HOST tensors."""
    import torch
    assert X.is_cuda and X.dtype == torch.float32 and X.dim() == 2 and X.stride(1) == 1
    m = _masks(masks)
    N, n_feat = X.shape
    out = dict(out or {})

    def pinned(shape, dtype):
        return torch.empty(shape, dtype=dtype, pin_memory=True)

    if lists:
        out.setdefault("idx", pinned((len(m), N, k), torch.int32))
        out.setdefault("dist", pinned((len(m), N, k), torch.float32))
    if scores:
        out.setdefault("kth", pinned((len(m), N), torch.float32))
        out.setdefault("mean", pinned((len(m), N), torch.float32))
        out.setdefault("indeg", pinned((len(m), N), torch.int32))
    for n, t in out.items():
        assert n.startswith("_") or t.is_pinned(), n
    ws = workspace if workspace is not None else _workspace(
        X, len(m), k, extra=stream_ring_bytes(N, k, masks_per_batch))
    _check(lib().snaps_knn_selfjoin_streamed(
        _dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m), k,
        masks_per_batch, _dptr(out.get("idx")), _dptr(out.get("dist")), _dptr(out.get("kth")),
        _dptr(out.get("mean")), _dptr(out.get("indeg")), _dptr(ws), ws.numel(), _stream(stream)))
    out["_workspace"] = ws
    return out


def knn_selfjoin_host(X_host, masks, k, masks_per_batch=None, *, lists=False, scores=True, out=None,
                      workspace=None, x_device=None, stream=None):
    """End-to-end call with HOST buffers: pinned X -> device, join, pinned host outputs.
    Returns the dict of pinned host tensors after the work is enqueued (caller synchronises).
    `out`, `workspace` and `x_device` may supply preallocated buffers for repeated calls."""
    import torch
    Xh = torch.as_tensor(X_host)
    if not Xh.is_pinned():
        Xh = Xh.pin_memory()
    s = torch.cuda.current_stream() if stream is None else stream
    with torch.cuda.stream(s):
        if x_device is None:
            Xd = Xh.to("cuda", non_blocking=True)
        else:
            Xd = x_device
            Xd.copy_(Xh, non_blocking=True)
    n_masks = len(_masks(masks))
    mpb = masks_per_batch or max(1, min(n_masks, 2048))
    out = knn_selfjoin_streamed(Xd, masks, k, mpb, lists=lists, scores=scores, out=out,
                                workspace=workspace, stream=s)
    out["_X"] = Xd
    return out


def probe_fp32_rate(kind: int, stream=None) -> float:
    v = ctypes.c_double(0.0)
    _check(lib().snaps_probe_fp32_rate(kind, ctypes.byref(v), _stream(stream)))
    return float(v.value)


def profile_enable(on: bool = True) -> None:
    _check(lib().snaps_profile_enable(1 if on else 0))


def profile_last_kernel_ms():
    """-> (summed device ms of the last call's join-kernel launches, number of launches)."""
    ms, n = ctypes.c_float(0.0), ctypes.c_int(0)
    _check(lib().snaps_profile_last_kernel_ms(ctypes.byref(ms), ctypes.byref(n)))
    return float(ms.value), int(n.value)


METRIC_KINDS = {"dssj_count": 0, "dssj_mean": 1, "knn_indegree": 2, "knn_mean": 3, "knn_kth": 3}


def rank_scores(metric: str, values, counts=None, *, ranks=True, order=True, stream=None):
    """snaps_rank_scores on a CUDA tensor values [n_rows, N] -> dict rank / order (int32)."""
    import torch
    assert values.is_cuda and values.dim() == 2 and values.is_contiguous()
    n_rows, N = values.shape
    out = {}
    if ranks:
        out["rank"] = torch.empty((n_rows, N), dtype=torch.int32, device=values.device)
    if order:
        out["order"] = torch.empty((n_rows, N), dtype=torch.int32, device=values.device)
    ws = torch.empty(int(lib().snaps_rank_workspace_bytes(N, n_rows)), dtype=torch.uint8, device=values.device)
    _check(lib().snaps_rank_scores(METRIC_KINDS[metric], _dptr(values), _dptr(counts), N, n_rows,
                                   _dptr(out.get("rank")), _dptr(out.get("order")), _dptr(ws), ws.numel(),
                                   _stream(stream)))
    out["_workspace"] = ws
    return out


def topn_overlap(order_a, order_b, n: int, stream=None):
    """snaps_topn_overlap (Eq. 2) -> fp32 tensor [n_rows]."""
    import torch
    n_rows, N = order_a.shape
    f = torch.empty(n_rows, dtype=torch.float32, device=order_a.device)
    _check(lib().snaps_topn_overlap(_dptr(order_a), _dptr(order_b), N, n_rows, n, _dptr(f), _stream(stream)))
    return f


def select_parameter(u_min, u_max, n_top: int = 0, stream=None):
    """snaps_select_parameter (Eq. 3): u_* [G, n_rows] fp32 -> int32 [n_rows]."""
    import torch
    G, n_rows = u_min.shape
    j = torch.empty(n_rows, dtype=torch.int32, device=u_min.device)
    _check(lib().snaps_select_parameter(_dptr(u_min), _dptr(u_max), G, n_rows, n_top, _dptr(j), _stream(stream)))
    return j


def knn_scores_at_k(knn_idx, knn_dist, k_j: int, stream=None):
    """snaps_knn_scores_at_k: lists [n_masks, N, k_max] -> dict kth / mean / indeg for k_j."""
    import torch
    n_masks, N, k_max = knn_dist.shape
    dev = knn_dist.device
    out = {"kth": torch.empty((n_masks, N), dtype=torch.float32, device=dev),
           "mean": torch.empty((n_masks, N), dtype=torch.float32, device=dev),
           "indeg": torch.empty((n_masks, N), dtype=torch.int32, device=dev)}
    _check(lib().snaps_knn_scores_at_k(N, n_masks, k_max, k_j, _dptr(knn_idx), _dptr(knn_dist),
                                       _dptr(out["kth"]), _dptr(out["mean"]), _dptr(out["indeg"]), _stream(stream)))
    return out


def range_selfjoin_grid(X, masks, eps_grid, *, sums=True, stream=None):
    """snaps_range_selfjoin_grid: eps_grid [n_masks, G] ascending per mask -> dict count / sumdist /
    mean, each [n_masks, G, N]."""
    import torch
    assert X.is_cuda and X.dtype == torch.float32 and X.dim() == 2 and X.stride(1) == 1
    m = _masks(masks)
    e = np.ascontiguousarray(np.asarray(eps_grid, dtype=np.float32))
    assert e.ndim == 2 and e.shape[0] == len(m)
    G = e.shape[1]
    N, n_feat = X.shape
    dev = X.device
    out = {"count": torch.empty((len(m), G, N), dtype=torch.int32, device=dev)}
    if sums:
        out["sumdist"] = torch.empty((len(m), G, N), dtype=torch.float32, device=dev)
        out["mean"] = torch.empty((len(m), G, N), dtype=torch.float32, device=dev)
    nbytes = int(lib().snaps_range_grid_workspace_bytes(N, n_feat, len(m), G))
    if nbytes == 0:
        raise SnapsError(1, "invalid sizes for the radius-grid workspace")
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    _check(lib().snaps_range_selfjoin_grid(
        _dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m),
        e.ctypes.data_as(ctypes.c_void_p), G, _dptr(out["count"]), _dptr(out.get("sumdist")),
        _dptr(out.get("mean")), _dptr(ws), ws.numel(), _stream(stream)))
    out["_workspace"] = ws
    return out


def knn_select_k(knn_idx, knn_dist, k_grid, n_top: int, stream=None):
    """snaps_knn_select_k: lists [n_masks, N, k_max] -> dict j_indeg / j_mean (grid index per mask)
    and u [4, G, n_masks] (U_min, U_max of the in-degree metric, then of the mean-distance metric)."""
    import torch
    n_masks, N, k_max = knn_dist.shape
    grid = np.ascontiguousarray(np.asarray(k_grid, dtype=np.int32))
    G = len(grid)
    dev = knn_dist.device
    out = {"j_indeg": torch.empty(n_masks, dtype=torch.int32, device=dev),
           "j_mean": torch.empty(n_masks, dtype=torch.int32, device=dev),
           "u": torch.empty((4, G, n_masks), dtype=torch.float32, device=dev)}
    ws = torch.empty(int(lib().snaps_select_k_workspace_bytes(N, n_masks)), dtype=torch.uint8, device=dev)
    _check(lib().snaps_knn_select_k(N, n_masks, k_max, _dptr(knn_idx), _dptr(knn_dist),
                                    grid.ctypes.data_as(ctypes.c_void_p), G, n_top, _dptr(out["j_indeg"]),
                                    _dptr(out["j_mean"]), _dptr(out["u"]), _dptr(ws), ws.numel(), _stream(stream)))
    out["_workspace"] = ws
    return out


def sample_distance_histogram(X, masks, sample_q, sample_c, rmax, n_bins: int, stream=None):
    """snaps_sample_distance_histogram -> int64 CUDA tensor [n_masks, n_bins]."""
    import torch
    m = _masks(masks)
    q = np.ascontiguousarray(np.asarray(sample_q, dtype=np.int32))
    c = np.ascontiguousarray(np.asarray(sample_c, dtype=np.int32))
    r = np.ascontiguousarray(np.asarray(rmax, dtype=np.float32))
    N, n_feat = X.shape
    hist = torch.empty((len(m), n_bins), dtype=torch.int64, device=X.device)
    ws = torch.empty(int(lib().snaps_dist_hist_workspace_bytes(len(q), len(c), len(m))), dtype=torch.uint8, device=X.device)
    _check(lib().snaps_sample_distance_histogram(
        _dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m),
        q.ctypes.data_as(ctypes.c_void_p), len(q), c.ctypes.data_as(ctypes.c_void_p), len(c),
        r.ctypes.data_as(ctypes.c_void_p), n_bins, _dptr(hist), _dptr(ws), ws.numel(), _stream(stream)))
    return hist


def eps_from_histogram(hist_host, rmax, N: int, pairs_per_mask: int, target_s: float) -> np.ndarray:
    """snaps_eps_from_histogram on a host copy of the histogram -> fp32 [n_masks]."""
    h = np.ascontiguousarray(np.asarray(hist_host, dtype=np.uint64))
    r = np.ascontiguousarray(np.asarray(rmax, dtype=np.float32))
    eps = np.empty(h.shape[0], dtype=np.float32)
    _check(lib().snaps_eps_from_histogram(h.ctypes.data_as(ctypes.c_void_p), h.shape[0], h.shape[1],
                                          r.ctypes.data_as(ctypes.c_void_p), N, pairs_per_mask, float(target_s),
                                          eps.ctypes.data_as(ctypes.c_void_p)))
    return eps
