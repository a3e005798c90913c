"""snaps-b200: the SNAPS (arXiv 2405.20176) kNN / eps self-joins and outlier scores for every
feature subspace, as hand-written sm_100a CUDA kernels behind a C ABI (include/snaps.h).

This package is the thin Python binding: argument marshalling only.  Every step of the path
runs in libsnaps.so's kernels; there is no CPU fallback -- importing works without a GPU (so
the symbol table can be checked), calling a join without the library or a device raises.
"""
from .binding import (  # noqa: F401
    SnapsError, lib, lib_path, version, workspace_bytes, stream_ring_bytes, planned_evals,
    knn_selfjoin, knn_selfjoin_static, STATIC_MAX_N, STATIC_MAX_MASKS, range_selfjoin, outlier_scores, knn_selfjoin_streamed, probe_fp32_rate,
    knn_selfjoin_host, knn_selfjoin_sink, range_selfjoin_sink, sink_batch_bytes, EXPORTED_SYMBOLS, ENGINES, profile_enable, profile_last_kernel_ms,
    range_selfjoin_grid, knn_select_k, eps_search, eps_for_selectivity, range_select_eps, range_from_knn, sample_distance_histogram, eps_from_histogram, rank_scores, topn_overlap, select_parameter, knn_scores_at_k, METRIC_KINDS,
)
