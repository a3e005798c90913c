"""ctypes binding for libsnaps.so -- same names as include/snaps.h, marshalling only."""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

EXPORTED_SYMBOLS = [
    "snaps_last_error", "snaps_version", "snaps_workspace_bytes", "snaps_planned_evals",
    "snaps_knn_selfjoin", "snaps_knn_selfjoin_static", "snaps_range_selfjoin", "snaps_outlier_scores",
    "snaps_stream_ring_bytes", "snaps_knn_selfjoin_streamed", "snaps_sink_batch_bytes",
    "snaps_knn_selfjoin_sink", "snaps_range_selfjoin_sink", "snaps_probe_fp32_rate",
    "snaps_profile_enable", "snaps_profile_last_kernel_ms",
    "snaps_rank_workspace_bytes", "snaps_rank_scores", "snaps_topn_overlap", "snaps_select_parameter",
    "snaps_knn_scores_at_k", "snaps_range_grid_workspace_bytes", "snaps_range_selfjoin_grid",
    "snaps_select_k_workspace_bytes", "snaps_knn_select_k",
    "snaps_dist_hist_workspace_bytes", "snaps_sample_distance_histogram", "snaps_eps_from_histogram",
    "snaps_eps_search_workspace_bytes", "snaps_eps_search",
    "snaps_select_eps_workspace_bytes", "snaps_range_select_eps", "snaps_range_from_knn",
]

ENGINES = {"auto": 0, "lattice": 1, "grid": 2}
FLAG_X_ON_HOST = 8
OUT_BITS = {"idx": 1, "dist": 2, "kth": 4, "mean": 8, "indeg": 16, "count": 32, "sumdist": 64, "eps_mean": 128}

_lib = None


class SnapsError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"snaps status {status}: {message}")
        self.status = status


class BatchView(ctypes.Structure):
    """snaps_batch_view of include/snaps.h."""
    _fields_ = [("mask_begin", ctypes.c_int), ("mask_end", ctypes.c_int),
                ("q_begin", ctypes.c_int64), ("q_end", ctypes.c_int64), ("N", ctypes.c_int64), ("k", ctypes.c_int),
                ("idx", ctypes.c_void_p), ("dist", ctypes.c_void_p), ("kth", ctypes.c_void_p),
                ("mean", ctypes.c_void_p), ("indeg", ctypes.c_void_p), ("count", ctypes.c_void_p),
                ("sumdist", ctypes.c_void_p), ("eps_mean", ctypes.c_void_p)]


BATCH_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.POINTER(BatchView))


class BatchSink(ctypes.Structure):
    """snaps_batch_sink of include/snaps.h."""
    _fields_ = [("h_buffers", ctypes.POINTER(ctypes.c_void_p)), ("n_buffers", ctypes.c_int),
                ("buffer_bytes", ctypes.c_size_t), ("want", ctypes.c_uint), ("consume", BATCH_FN),
                ("user", ctypes.c_void_p)]


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
        L.snaps_workspace_bytes.argtypes = [i64, i32, i32, i32, i32]
        L.snaps_planned_evals.restype = i64
        L.snaps_planned_evals.argtypes = [i64, i32, vp, i32]
        L.snaps_knn_selfjoin.restype = i32
        L.snaps_knn_selfjoin.argtypes = [vp, i64, i32, i64, vp, i32, i32, i64, i64, i32, vp, vp, vp, vp, vp, vp, sz, vp]
        L.snaps_knn_selfjoin_static.restype = i32
        L.snaps_knn_selfjoin_static.argtypes = [vp, i64, i32, i64, vp, i32, i32, vp, vp, vp, vp, vp, vp]
        L.snaps_range_selfjoin.restype = i32
        L.snaps_range_selfjoin.argtypes = [vp, i64, i32, i64, vp, i32, vp, i64, i64, i32, vp, vp, vp, vp, sz, vp]
        L.snaps_outlier_scores.restype = i32
        L.snaps_outlier_scores.argtypes = [i64, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.snaps_stream_ring_bytes.restype = sz
        L.snaps_stream_ring_bytes.argtypes = [i64, i64, i32, i32]
        L.snaps_knn_selfjoin_streamed.restype = i32
        L.snaps_knn_selfjoin_streamed.argtypes = [vp, i64, i32, i64, vp, i32, i32, i32, i64, i64, i32,
                                                  vp, vp, vp, vp, vp, vp, sz, vp]
        L.snaps_sink_batch_bytes.restype = sz
        L.snaps_sink_batch_bytes.argtypes = [i64, i64, i32, i32, ctypes.c_uint]
        L.snaps_knn_selfjoin_sink.restype = i32
        L.snaps_knn_selfjoin_sink.argtypes = [vp, i64, i32, i64, vp, i32, i32, i32, i64, i64, i32,
                                              ctypes.POINTER(BatchSink), vp, sz, vp]
        L.snaps_range_selfjoin_sink.restype = i32
        L.snaps_range_selfjoin_sink.argtypes = [vp, i64, i32, i64, vp, i32, vp, i32, i64, i64, i32,
                                                ctypes.POINTER(BatchSink), vp, sz, vp]
        L.snaps_probe_fp32_rate.restype = i32
        L.snaps_probe_fp32_rate.argtypes = [i32, ctypes.POINTER(ctypes.c_double), vp, vp]
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
        L.snaps_range_grid_workspace_bytes.argtypes = [i64, i32, i32, i32, i32]
        L.snaps_range_selfjoin_grid.restype = i32
        L.snaps_range_selfjoin_grid.argtypes = [vp, i64, i32, i64, vp, i32, vp, i32, i64, i64, i32, vp, vp, vp, vp, sz, vp]
        L.snaps_dist_hist_workspace_bytes.restype = sz
        L.snaps_dist_hist_workspace_bytes.argtypes = [i32, i32, i32]
        L.snaps_sample_distance_histogram.restype = i32
        L.snaps_sample_distance_histogram.argtypes = [vp, i64, i32, i64, vp, i32, vp, i32, vp, i32, vp, i32, vp, vp, sz, vp]
        L.snaps_eps_from_histogram.restype = i32
        L.snaps_eps_from_histogram.argtypes = [vp, i32, i32, vp, i64, i64, ctypes.c_double, vp]
        L.snaps_eps_search_workspace_bytes.restype = sz
        L.snaps_eps_search_workspace_bytes.argtypes = [i32, i32, i32, i32, i32]
        L.snaps_eps_search.restype = i32
        L.snaps_eps_search.argtypes = [vp, i64, i32, i64, vp, i32, vp, i32, vp, i32, i32, vp, i32, vp, vp, vp, vp, sz, vp]
        L.snaps_select_eps_workspace_bytes.restype = sz
        L.snaps_select_eps_workspace_bytes.argtypes = [i64, i32, i32, i32, i32, i32, i32, i32]
        L.snaps_range_select_eps.restype = i32
        L.snaps_range_select_eps.argtypes = [vp, i64, i32, i64, vp, i32, vp, i32, vp, i32, i32, ctypes.c_double,
                                             ctypes.c_double, i32, i32, i32, vp, vp, vp, vp, vp, sz, vp]
        L.snaps_range_from_knn.restype = i32
        L.snaps_range_from_knn.argtypes = [i64, i32, i32, vp, vp, vp, vp, vp, vp, vp]
        L.snaps_select_k_workspace_bytes.restype = sz
        L.snaps_select_k_workspace_bytes.argtypes = [i64, i32, i32]
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


def _flags(engine: str, x_on_host: bool = False) -> int:
    return ENGINES[engine] | (FLAG_X_ON_HOST if x_on_host else 0)


def _qrange(q_range, N):
    return (0, N) if q_range is None else (int(q_range[0]), int(q_range[1]))


def workspace_bytes(N: int, n_feat: int, n_masks: int, k: int, engine: str = "auto", x_on_host: bool = False) -> int:
    return int(lib().snaps_workspace_bytes(N, n_feat, n_masks, k, _flags(engine, x_on_host)))


def stream_ring_bytes(nq: int, N: int, k: int, masks_per_batch: int) -> int:
    return int(lib().snaps_stream_ring_bytes(nq, N, k, masks_per_batch))


def planned_evals(N: int, n_feat: int, masks) -> int:
    m = _masks(masks)
    return int(lib().snaps_planned_evals(N, n_feat, m.ctypes.data_as(ctypes.c_void_p), len(m)))


def _workspace(N, n_feat, n_masks, k, device, engine="auto", extra=0, x_on_host=False):
    import torch
    nbytes = workspace_bytes(N, n_feat, n_masks, k, engine, x_on_host)
    if nbytes == 0:
        raise SnapsError(1, "invalid sizes for workspace")
    return torch.empty(nbytes + extra, dtype=torch.uint8, device=device)


def knn_selfjoin(X, masks, k, *, lists=True, scores=True, out=None, workspace=None, stream=None,
                 q_range=None, engine="auto"):
    """snaps_knn_selfjoin on a CUDA fp32 tensor X [N, n_feat].

    Returns a dict with idx/dist [n_masks, nq, k] (if lists), kth/mean [n_masks, nq] and indeg
    [n_masks, N] (if scores), all torch CUDA tensors; nq = q_range[1] - q_range[0] (default: all N
    objects are queries).  `out` may supply preallocated tensors by those names."""
    import torch
    assert X.is_cuda and X.dtype == torch.float32 and X.dim() == 2 and X.stride(1) == 1
    m = _masks(masks)
    N, n_feat = X.shape
    q0, q1 = _qrange(q_range, N)
    nq = q1 - q0
    out = dict(out or {})
    dev = X.device
    if lists:
        out.setdefault("idx", torch.empty((len(m), nq, k), dtype=torch.int32, device=dev))
        out.setdefault("dist", torch.empty((len(m), nq, k), dtype=torch.float32, device=dev))
    if scores:
        out.setdefault("kth", torch.empty((len(m), nq), dtype=torch.float32, device=dev))
        out.setdefault("mean", torch.empty((len(m), nq), dtype=torch.float32, device=dev))
        out.setdefault("indeg", torch.empty((len(m), N), dtype=torch.int32, device=dev))
    ws = workspace if workspace is not None else _workspace(N, n_feat, len(m), k, dev, engine)
    _check(lib().snaps_knn_selfjoin(
        _dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m), k, q0, q1, _flags(engine),
        _dptr(out.get("idx")), _dptr(out.get("dist")), _dptr(out.get("kth")),
        _dptr(out.get("mean")), _dptr(out.get("indeg")), _dptr(ws), ws.numel(), _stream(stream)))
    out["_workspace"] = ws
    return out


STATIC_MAX_N = 32768          # SNAPS_STATIC_MAX_N
STATIC_MAX_MASKS = 2048       # SNAPS_STATIC_MAX_MASKS


def knn_selfjoin_static(X, masks, k, *, lists=True, scores=True, out=None, stream=None):
    """snaps_knn_selfjoin_static: the kNN self-join with the library's built-in scratch array instead
    of a workspace (the C call allocates nothing on the device; N <= 32,768, n_masks <= 2,048,
    k <= 32; calls that overlap on one GPU race).  Outputs as knn_selfjoin; pass them in `out` to keep
    this wrapper from allocating them."""
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
    _check(lib().snaps_knn_selfjoin_static(
        _dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m), k,
        _dptr(out.get("idx")), _dptr(out.get("dist")), _dptr(out.get("kth")),
        _dptr(out.get("mean")), _dptr(out.get("indeg")), _stream(stream)))
    return out


def range_selfjoin(X, masks, eps, *, sums=True, out=None, workspace=None, stream=None, q_range=None,
                   engine="auto"):
    """snaps_range_selfjoin: returns dict count [n_masks, nq] (int32 view of uint32) and, if
    sums, sumdist / mean."""
    import torch
    assert X.is_cuda and X.dtype == torch.float32 and X.dim() == 2 and X.stride(1) == 1
    m = _masks(masks)
    e = np.ascontiguousarray(np.asarray(eps, dtype=np.float32).ravel())
    assert len(e) == len(m)
    N, n_feat = X.shape
    q0, q1 = _qrange(q_range, N)
    nq = q1 - q0
    out = dict(out or {})
    dev = X.device
    out.setdefault("count", torch.empty((len(m), nq), dtype=torch.int32, device=dev))
    if sums:
        out.setdefault("sumdist", torch.empty((len(m), nq), dtype=torch.float32, device=dev))
        out.setdefault("mean", torch.empty((len(m), nq), dtype=torch.float32, device=dev))
    ws = workspace if workspace is not None else _workspace(N, n_feat, len(m), 0, dev, engine)
    _check(lib().snaps_range_selfjoin(
        _dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m),
        e.ctypes.data_as(ctypes.c_void_p), q0, q1, _flags(engine), _dptr(out["count"]), _dptr(out.get("sumdist")),
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
                          workspace=None, stream=None, q_range=None, engine="auto", x_on_host=False):
    """snaps_knn_selfjoin_streamed: outputs land in PINNED HOST tensors.  With x_on_host, X is a host
    tensor (pinned or pageable) and the copy to the device is part of the call."""
    import torch
    assert X.dtype == torch.float32 and X.dim() == 2 and X.stride(1) == 1
    assert X.is_cuda != bool(x_on_host)
    m = _masks(masks)
    N, n_feat = X.shape
    q0, q1 = _qrange(q_range, N)
    nq = q1 - q0
    out = dict(out or {})

    def pinned(shape, dtype):
        return torch.empty(shape, dtype=dtype, pin_memory=True)

    if lists:
        out.setdefault("idx", pinned((len(m), nq, k), torch.int32))
        out.setdefault("dist", pinned((len(m), nq, k), torch.float32))
    if scores:
        out.setdefault("kth", pinned((len(m), nq), torch.float32))
        out.setdefault("mean", pinned((len(m), nq), torch.float32))
        out.setdefault("indeg", pinned((len(m), N), torch.int32))
    for n, t in out.items():
        assert n.startswith("_") or t.is_pinned(), n
    dev = X.device if X.is_cuda else torch.device("cuda", torch.cuda.current_device())
    ws = workspace if workspace is not None else _workspace(
        N, n_feat, len(m), k, dev, engine, extra=stream_ring_bytes(nq, N, k, masks_per_batch), x_on_host=x_on_host)
    _check(lib().snaps_knn_selfjoin_streamed(
        _dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m), k,
        masks_per_batch, q0, q1, _flags(engine, x_on_host), _dptr(out.get("idx")), _dptr(out.get("dist")),
        _dptr(out.get("kth")), _dptr(out.get("mean")), _dptr(out.get("indeg")), _dptr(ws), ws.numel(),
        _stream(stream)))
    out["_workspace"] = ws
    return out


def knn_selfjoin_host(X_host, masks, k, masks_per_batch=None, *, lists=False, scores=True, out=None,
                      workspace=None, stream=None, engine="auto"):
    """End-to-end call with HOST buffers only: ONE C call (snaps_knn_selfjoin_streamed with
    SNAPS_FLAG_X_ON_HOST) copies the pinned table to the device, joins, and copies the outputs into
    pinned host tensors.  Returns them after the work is enqueued (caller synchronises)."""
    import torch
    Xh = torch.as_tensor(X_host)
    if not Xh.is_pinned():
        Xh = Xh.pin_memory()
    n_masks = len(_masks(masks))
    mpb = masks_per_batch or max(1, min(n_masks, 2048))
    out = knn_selfjoin_streamed(Xh, masks, k, mpb, lists=lists, scores=scores, out=out, workspace=workspace,
                                stream=stream, engine=engine, x_on_host=True)
    out["_X"] = Xh
    return out


def sink_batch_bytes(nq: int, N: int, k: int, masks_per_batch: int, want) -> int:
    bits = sum(OUT_BITS[w] for w in want)
    return int(lib().snaps_sink_batch_bytes(nq, N, k, masks_per_batch, bits))


def _run_sink(kind, X, masks, k, eps, masks_per_batch, want, consume, n_buffers, q_range, engine, workspace, stream):
    import torch
    assert X.is_cuda and X.dtype == torch.float32 and X.dim() == 2 and X.stride(1) == 1
    m = _masks(masks)
    N, n_feat = X.shape
    q0, q1 = _qrange(q_range, N)
    nq = q1 - q0
    bits = sum(OUT_BITS[w] for w in want)
    nbytes = int(lib().snaps_sink_batch_bytes(nq, N, k, masks_per_batch, bits))
    bufs = [torch.empty(nbytes, dtype=torch.uint8, pin_memory=True) for _ in range(n_buffers)]
    ptrs = (ctypes.c_void_p * n_buffers)(*[b.data_ptr() for b in bufs])
    shapes = {"idx": (nq, k), "dist": (nq, k), "kth": (nq,), "mean": (nq,), "indeg": (N,),
              "count": (nq,), "sumdist": (nq,), "eps_mean": (nq,)}
    dtypes = {"idx": np.int32, "dist": np.float32, "kth": np.float32, "mean": np.float32, "indeg": np.int32,
              "count": np.uint32, "sumdist": np.float32, "eps_mean": np.float32}
    errors = []

    def trampoline(_user, view_p):
        v = view_p.contents
        nm = v.mask_end - v.mask_begin
        arrays = {}
        for name in shapes:
            addr = getattr(v, name)
            if addr:
                shp = (nm,) + shapes[name]
                n_el = int(np.prod(shp))
                buf = (ctypes.c_byte * (n_el * 4)).from_address(addr)
                arrays[name] = np.frombuffer(buf, dtype=dtypes[name], count=n_el).reshape(shp)
        try:
            consume(v.mask_begin, v.mask_end, arrays)
        except Exception as e:          # a Python exception must not unwind through the C frames
            errors.append(e)

    cb = BATCH_FN(trampoline)
    sink = BatchSink(ptrs, n_buffers, nbytes, bits, cb, None)
    ws = workspace if workspace is not None else _workspace(
        N, n_feat, len(m), k, X.device, engine, extra=stream_ring_bytes(nq, N, k, masks_per_batch))
    if kind == "knn":
        rc = lib().snaps_knn_selfjoin_sink(_dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m), k,
                                           masks_per_batch, q0, q1, _flags(engine), ctypes.byref(sink), _dptr(ws),
                                           ws.numel(), _stream(stream))
    else:
        e = np.ascontiguousarray(np.asarray(eps, dtype=np.float32).ravel())
        assert len(e) == len(m)
        rc = lib().snaps_range_selfjoin_sink(_dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m),
                                             e.ctypes.data_as(ctypes.c_void_p), masks_per_batch, q0, q1, _flags(engine),
                                             ctypes.byref(sink), _dptr(ws), ws.numel(), _stream(stream))
    _check(rc)
    if errors:
        raise errors[0]
    return ws


def knn_selfjoin_sink(X, masks, k, masks_per_batch, consume, *, want=("kth", "mean", "indeg"), n_buffers=2,
                      q_range=None, engine="auto", workspace=None, stream=None):
    """snaps_knn_selfjoin_sink: `consume(mask_begin, mask_end, arrays)` is called once per mask group
    with numpy views into a recycled pinned host buffer (valid only during the call)."""
    return _run_sink("knn", X, masks, k, None, masks_per_batch, want, consume, n_buffers, q_range, engine, workspace, stream)


def range_selfjoin_sink(X, masks, eps, masks_per_batch, consume, *, want=("count", "sumdist", "eps_mean"), n_buffers=2,
                        q_range=None, engine="auto", workspace=None, stream=None):
    """snaps_range_selfjoin_sink, see knn_selfjoin_sink."""
    return _run_sink("range", X, masks, 0, eps, masks_per_batch, want, consume, n_buffers, q_range, engine, workspace, stream)


def probe_fp32_rate(kind: int, stream=None) -> float:
    import torch
    v = ctypes.c_double(0.0)
    scratch = torch.empty(4096, dtype=torch.uint8, device="cuda")
    _check(lib().snaps_probe_fp32_rate(kind, ctypes.byref(v), _dptr(scratch), _stream(stream)))
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


def range_selfjoin_grid(X, masks, eps_grid, *, sums=True, stream=None, q_range=None, engine="auto"):
    """snaps_range_selfjoin_grid: eps_grid [n_masks, G] ascending per mask -> dict count / sumdist /
    mean, each [n_masks, G, nq]."""
    import torch
    assert X.is_cuda and X.dtype == torch.float32 and X.dim() == 2 and X.stride(1) == 1
    m = _masks(masks)
    e = np.ascontiguousarray(np.asarray(eps_grid, dtype=np.float32))
    assert e.ndim == 2 and e.shape[0] == len(m)
    G = e.shape[1]
    N, n_feat = X.shape
    q0, q1 = _qrange(q_range, N)
    nq = q1 - q0
    dev = X.device
    out = {"count": torch.empty((len(m), G, nq), dtype=torch.int32, device=dev)}
    if sums:
        out["sumdist"] = torch.empty((len(m), G, nq), dtype=torch.float32, device=dev)
        out["mean"] = torch.empty((len(m), G, nq), dtype=torch.float32, device=dev)
    nbytes = int(lib().snaps_range_grid_workspace_bytes(N, n_feat, len(m), G, _flags(engine)))
    if nbytes == 0:
        raise SnapsError(1, "invalid sizes for the radius-grid workspace")
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    _check(lib().snaps_range_selfjoin_grid(
        _dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m),
        e.ctypes.data_as(ctypes.c_void_p), G, q0, q1, _flags(engine), _dptr(out["count"]), _dptr(out.get("sumdist")),
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
    ws = torch.empty(int(lib().snaps_select_k_workspace_bytes(N, n_masks, G)), dtype=torch.uint8, device=dev)
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


def eps_search(X, masks, sample_q, sample_c, targets, n_bins: int = 4096, *, hist=False, stream=None):
    """snaps_eps_search -> dict eps_mean [n_masks], eps [n_masks, n_targets] (CUDA fp32) and, if asked,
    hist [n_masks, n_bins] (int64)."""
    import torch
    m = _masks(masks)
    q = np.ascontiguousarray(np.asarray(sample_q, dtype=np.int32))
    c = np.ascontiguousarray(np.asarray(sample_c, dtype=np.int32))
    t = np.ascontiguousarray(np.asarray(targets, dtype=np.float64).ravel())
    N, n_feat = X.shape
    dev = X.device
    out = {"eps_mean": torch.empty(len(m), dtype=torch.float32, device=dev),
           "eps": torch.empty((len(m), len(t)), dtype=torch.float32, device=dev)}
    if hist:
        out["hist"] = torch.empty((len(m), n_bins), dtype=torch.int64, device=dev)
    ws = torch.empty(int(lib().snaps_eps_search_workspace_bytes(len(q), len(c), len(m), n_bins, len(t))),
                     dtype=torch.uint8, device=dev)
    _check(lib().snaps_eps_search(
        _dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m),
        q.ctypes.data_as(ctypes.c_void_p), len(q), c.ctypes.data_as(ctypes.c_void_p), len(c), n_bins,
        t.ctypes.data_as(ctypes.c_void_p), len(t), _dptr(out["eps_mean"]), _dptr(out["eps"]), _dptr(out.get("hist")),
        _dptr(ws), ws.numel(), _stream(stream)))
    out["_workspace"] = ws
    return out


def eps_for_selectivity(X, masks, target_neighbours: float, seed: int = 0, n_query_sample: int = 1000,
                        n_cand_sample: int = 100_000, n_bins: int = 8192) -> np.ndarray:
    """Radii for a target mean neighbour count from seeded samples (marshalling around snaps_eps_search:
    the sample ids are drawn here, the search runs on the device).  -> fp32 [n_masks] on the host."""
    N = X.shape[0]
    rng = np.random.default_rng(seed)
    q = np.sort(rng.choice(N, min(n_query_sample, N), replace=False))
    c = np.sort(rng.choice(N, min(n_cand_sample, N), replace=False))
    out = eps_search(X, masks, q, c, [target_neighbours], n_bins)
    return out["eps"][:, 0].cpu().numpy()


def range_select_eps(X, masks, sample_q, sample_c, s_min: float, s_max: float, G: int, n_top: int, n_bins: int = 4096,
                     *, engine="auto", stream=None):
    """snaps_range_select_eps -> dict eps_grid [n_masks, G], j_count / j_mean [n_masks] (grid index of the
    selected radius per DSSJ metric) and u [4, G, n_masks]."""
    import torch
    m = _masks(masks)
    q = np.ascontiguousarray(np.asarray(sample_q, dtype=np.int32))
    c = np.ascontiguousarray(np.asarray(sample_c, dtype=np.int32))
    N, n_feat = X.shape
    dev = X.device
    out = {"eps_grid": torch.empty((len(m), G), dtype=torch.float32, device=dev),
           "j_count": torch.empty(len(m), dtype=torch.int32, device=dev),
           "j_mean": torch.empty(len(m), dtype=torch.int32, device=dev),
           "u": torch.empty((4, G, len(m)), dtype=torch.float32, device=dev)}
    nbytes = int(lib().snaps_select_eps_workspace_bytes(N, n_feat, len(m), G, len(q), len(c), n_bins, _flags(engine)))
    if nbytes == 0:
        raise SnapsError(1, "invalid sizes for the eps selection workspace")
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    _check(lib().snaps_range_select_eps(
        _dptr(X), N, n_feat, X.stride(0), m.ctypes.data_as(ctypes.c_void_p), len(m),
        q.ctypes.data_as(ctypes.c_void_p), len(q), c.ctypes.data_as(ctypes.c_void_p), len(c), n_bins,
        float(s_min), float(s_max), G, n_top, _flags(engine), _dptr(out["eps_grid"]), _dptr(out["j_count"]),
        _dptr(out["j_mean"]), _dptr(out["u"]), _dptr(ws), ws.numel(), _stream(stream)))
    out["_workspace"] = ws
    return out


def range_from_knn(knn_dist, eps, stream=None):
    """snaps_range_from_knn: lists [n_masks, nq, k] (CUDA fp32) + radii [n_masks] (CUDA fp32 or array-like) ->
    dict count (int32 view) / sumdist / mean [n_masks, nq] and complete (uint8: 1 = the list holds the whole
    eps-neighbourhood)."""
    import torch
    n_masks, nq, k = knn_dist.shape
    dev = knn_dist.device
    e = eps if hasattr(eps, "is_cuda") else torch.as_tensor(np.asarray(eps, dtype=np.float32))
    e = e.to(device=dev, dtype=torch.float32).contiguous()
    assert e.numel() == n_masks and knn_dist.is_contiguous()
    out = {"count": torch.empty((n_masks, nq), dtype=torch.int32, device=dev),
           "sumdist": torch.empty((n_masks, nq), dtype=torch.float32, device=dev),
           "mean": torch.empty((n_masks, nq), dtype=torch.float32, device=dev),
           "complete": torch.empty((n_masks, nq), dtype=torch.uint8, device=dev)}
    _check(lib().snaps_range_from_knn(nq, n_masks, k, _dptr(knn_dist), _dptr(e), _dptr(out["count"]),
                                      _dptr(out["sumdist"]), _dptr(out["mean"]), _dptr(out["complete"]), _stream(stream)))
    return out
