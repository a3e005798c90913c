/*
 * snaps.h -- C ABI of libsnaps: the data-parallel hot path of SNAPS population
 * outlier detection (arXiv 2405.20176) on one B200 (sm_100a).
 *
 * Citations are lines of /root/reference/PAPER.md.  "Readings" A1..A19 are the
 * interpretations listed in DESIGN.md.
 *
 * Conventions for every entry point
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  Output
 *     pointers named out_* are device pointers unless stated otherwise.
 *   - The caller owns every buffer; the library allocates no device or pinned
 *     memory and never frees caller memory.  Scratch comes from d_workspace
 *     (size from snaps_workspace_bytes with the same N, n_feat, n_masks, k and
 *     flags).  The batched calls keep one side stream and a few events per
 *     calling thread, created on first use.  No environment variable or other
 *     process-global state changes what a call does.
 *   - All device work is enqueued on `stream` (a cudaStream_t passed as
 *     void*; NULL = the legacy default stream).  The call returns when the
 *     work is enqueued; host-side planning may block the calling thread but
 *     never synchronises the device.  "stream complete" => all outputs final.
 *   - Return value: SNAPS_OK or an error code; argument errors are detected
 *     before any launch.  snaps_last_error() gives a thread-local message.
 *   - X is row-major, N rows (objects), n_feat columns (features), row stride
 *     ld floats, fp32, normalised to [0,1] by the caller.  NaN
 *     in X is undefined behaviour (the paper removes NaNs first).
 *   - A subspace ("feature space") is a uint16 bitmask: bit j
 *     set <=> column j is used.  Masks must be non-zero with no bit >= n_feat.
 *   - Distances are Euclidean on the masked columns (reading A1), computed in
 *     fp32 by direct differences ("32-bit floating point").
 *   - Results do not depend on batching, tile sizes or scheduling; kNN ties
 *     are broken by the smaller object id (reading A3).
 */
#ifndef SNAPS_H
#define SNAPS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef int snaps_status;
#define SNAPS_OK 0
#define SNAPS_INVALID_ARG 1
#define SNAPS_CUDA_ERROR 2
#define SNAPS_WORKSPACE_TOO_SMALL 3
#define SNAPS_UNSUPPORTED 4

#define SNAPS_MAX_FEATURES 15 /* PAPER.md:109 "We examine d <= 15" */
#define SNAPS_MAX_K 4096       /* grid engine (k_max = 4096 on SNAPShot1; 256 on LSST5M).
                                  Lists up to 256 entries live in shared memory; longer ones are built in
                                  place in out_idx / out_dist, which must then both be given */
#define SNAPS_LATTICE_MAX_K 32 /* sub-lattice engine: lists live in shared memory */

/*
 * `flags` of the join entry points.  Bits 0..2 choose the engine:
 *   SNAPS_ENGINE_AUTO     sub-lattice engine for N < 2^18 and k <= 32, grid engine otherwise
 *   SNAPS_ENGINE_LATTICE  batches of 64 subspaces {H u T : T within features 0..5} share every
 *                         pair's squared differences; brute force with an exact filter.  For
 *                         mask lists with sub-lattice structure (all subsets) on L2-sized tables.
 *   SNAPS_ENGINE_GRID     one subspace at a time through a grid index on up to three of its
 *                         features.  For arbitrary mask lists, large N, k <= 4096.
 * Both engines compute the same joins; a pair's fp32 distance may differ in the last bit between
 * them (different summation order), so equal-distance ties may resolve differently.
 * SNAPS_FLAG_X_ON_HOST: the table pointer is a HOST pointer (pinned or pageable); the call copies
 * it into the workspace first (the copy is part of the enqueued work).
 * snaps_workspace_bytes must be given the same flags as the join that uses the workspace.
 */
#define SNAPS_ENGINE_AUTO 0
#define SNAPS_ENGINE_LATTICE 1
#define SNAPS_ENGINE_GRID 2
#define SNAPS_ENGINE_MASK 7
#define SNAPS_FLAG_X_ON_HOST 8

/* Message for the last non-OK status on this thread (static storage). */
const char *snaps_last_error(void);

/* Library version string (static storage). */
const char *snaps_version(void);

/*
 * Bytes of device scratch the joins need for these sizes and flags.  Sub-lattice engine: the
 * table staged twice (80-byte rows; 32-row blocks of four float4 groups) and batch descriptors.
 * Grid engine: staged rows, 4096 quantile edges and a 12-bit bin per object and feature, and one
 * subspace's index (sorted cell keys, permutation, cell starts, compact rows; ~110 bytes per
 * object).  k may be 0 for the range joins.  Returns 0 on invalid sizes.
 */
size_t snaps_workspace_bytes(int64_t N, int n_feat, int n_masks, int k, int flags);

/*
 * Number of (ordered query-candidate pair, mask) distance evaluations an
 * unpruned pass over the planned sub-lattice batches amounts to, INCLUDING the
 * lattice slots the planner enumerates but does not output (64 per batch); the
 * algorithmic count is N*N*n_masks.  The kernels reach the same result with
 * fewer operations (exact lower-bound filter).  Used by
 * bench.py's roofline arithmetic.  h_masks: host.
 */
int64_t snaps_planned_evals(int64_t N, int n_feat, const uint16_t *h_masks, int n_masks);

/*
 * kNN self-join, kNNSJ (section 3.6): for every mask S and
 * every query object i in [q_begin, q_end), the k objects j != i (of all N) with
 * the smallest (D(i,j;S), j).  Self is excluded by index (reading
 * A4): a different object at distance 0 is a neighbour.
 *
 *   d_X        device (host with SNAPS_FLAG_X_ON_HOST), [N][ld] fp32; every column finite,
 *              including columns no mask uses
 *   h_masks    host, [n_masks] uint16
 *   k          1 <= k <= min(N-1, SNAPS_MAX_K); the sub-lattice engine holds k <= 32; k > 256 needs
 *              out_idx and out_dist (the lists are built in place, or, for k > 384 on N <= 131,072 with the
 *              workspace snaps_workspace_bytes reports for that k, by radix selection: same lists, faster)
 *   q_begin, q_end   the queries: 0 <= q_begin < q_end <= N; nq = q_end - q_begin.  A rank of a
 *              multi-GPU run owns one slice (no exchange step);
 *              (0, N) is the whole self-join
 *   out_idx    device, [n_masks][nq][k] int32 neighbour ids, ascending by (distance, id); may be NULL
 *   out_dist   device, [n_masks][nq][k] fp32 distances D (not D^2), ascending; may be NULL
 *   out_kth    device, [n_masks][nq] fp32, D_(k): k-th-neighbour distance
 *              (BASELINE.json configs[0], reading A11); may be NULL
 *   out_mean   device, [n_masks][nq] fp32, (1/k) sum_r D_(r): the distance-aware
 *              kNN metric (reading A5); may be NULL
 *   out_indeg  device, [n_masks][N] int32, in-degree of the kNN graph restricted to the queries of
 *              this call: number of queries that list object j among their kNN, the
 *              distance-oblivious metric; summing the arrays of disjoint query
 *              slices gives the full in-degree; ZEROED by the call; may be NULL
 *
 * Scores-only operation (out_idx == out_dist == NULL) is supported because
 * the lists of the all-subspace run are 83 GB.  Errors: SNAPS_INVALID_ARG for
 * N < 2, n_feat outside 1..15, ld < n_feat, NULL d_X/h_masks, n_masks < 1, a
 * zero mask or a mask bit >= n_feat, k or the query range outside their ranges,
 * d_X not 4-byte aligned, all five outputs NULL, an unknown engine;
 * SNAPS_WORKSPACE_TOO_SMALL; SNAPS_CUDA_ERROR.
 */
snaps_status snaps_knn_selfjoin(const float *d_X, int64_t N, int n_feat, int64_t ld,
                                const uint16_t *h_masks, int n_masks, int k,
                                int64_t q_begin, int64_t q_end, int flags,
                                int32_t *out_idx, float *out_dist,
                                float *out_kth, float *out_mean, int32_t *out_indeg,
                                void *d_workspace, size_t workspace_bytes, void *stream);

/*
 * The same kNN self-join (scores of PAPER.md:251-252) for callers that cannot
 * allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): no workspace argument.  The staged copies of the table, the work counter and the batch
 * descriptors of the sub-lattice engine live in a fixed array of SNAPS_STATIC_SCRATCH_BYTES (5.8 MB)
 * inside the library, which every GPU that loads the library holds until the process exits.  The call
 * allocates nothing on the device (no cudaMalloc / cudaFree / allocating library routine).
 *
 * Arguments as snaps_knn_selfjoin with q_begin = 0, q_end = N, the sub-lattice engine, and
 *   N        2 <= N <= SNAPS_STATIC_MAX_N (32,768: SNAPShot1's 31,693 objects fit)
 *   n_masks  1 <= n_masks <= SNAPS_STATIC_MAX_MASKS (2,048)
 *   k        1 <= k <= min(N-1, SNAPS_LATTICE_MAX_K)
 *   d_X      device only.
 * Larger sizes are rejected with SNAPS_UNSUPPORTED and a message that names the limit; results are
 * identical to snaps_knn_selfjoin's (same kernels).  Every call on a device shares the one array: it
 * keeps the last call's contents (each call rewrites all it reads and zeroes the work counter), and
 * two calls that overlap on the same GPU -- different streams, different threads -- race; serialise them.
 */
#define SNAPS_STATIC_MAX_N 32768
#define SNAPS_STATIC_MAX_MASKS 2048
#define SNAPS_STATIC_SCRATCH_BYTES 5800192
snaps_status snaps_knn_selfjoin_static(const float *d_X, int64_t N, int n_feat, int64_t ld,
                                       const uint16_t *h_masks, int n_masks, int k,
                                       int32_t *out_idx, float *out_dist,
                                       float *out_kth, float *out_mean, int32_t *out_indeg,
                                       void *stream);

/*
 * eps range self-join, DSSJ (section 3.5): for
 * every mask S and query object i in [q_begin, q_end), the objects j != i with
 * D(i,j;S) <= eps_S (closed ball, reading A2; pairs within 1e-6 relative of eps
 * may fall on either side in fp32).
 *
 *   h_eps        host, [n_masks] fp32, each finite and > 0
 *   out_count    device, [n_masks][nq] uint32: number of neighbours within eps,
 *                self excluded = the distance-oblivious DSSJ
 *                metric; required
 *   out_sumdist  device, [n_masks][nq] fp32: sum of D over those neighbours
 *                (numerator of the distance-aware metric); may be
 *                NULL
 *   out_mean     device, [n_masks][nq] fp32: sumdist/count, 0 when count == 0
 *                (reading A6); may be NULL
 */
snaps_status snaps_range_selfjoin(const float *d_X, int64_t N, int n_feat, int64_t ld,
                                  const uint16_t *h_masks, int n_masks, const float *h_eps,
                                  int64_t q_begin, int64_t q_end, int flags,
                                  uint32_t *out_count, float *out_sumdist, float *out_mean,
                                  void *d_workspace, size_t workspace_bytes, void *stream);

/*
 * Per-object outlier scores from join outputs already on the device
 * (PAPER.md:164-165, 251-252).  Any input group and any output may be NULL.
 *
 *   knn_idx, knn_dist   [n_masks][N][k] as written by snaps_knn_selfjoin
 *   eps_count, eps_sumdist  [n_masks][N] as written by snaps_range_selfjoin
 *   out_kth, out_knn_mean   [n_masks][N] fp32 (need knn_dist)
 *   out_indegree            [n_masks][N] int32 (needs knn_idx); zeroed here
 *   out_eps_mean            [n_masks][N] fp32 = sumdist/count, 0 if count == 0
 */
snaps_status snaps_outlier_scores(int64_t N, int n_masks, int k,
                                  const int32_t *knn_idx, const float *knn_dist,
                                  const uint32_t *eps_count, const float *eps_sumdist,
                                  float *out_kth, float *out_knn_mean, int32_t *out_indegree,
                                  float *out_eps_mean, void *stream);

/*
 * kNN -> DSSJ reuse (the paper's future work: "providing the set of k nearest neighbors from
 * kNNSJ to DSSJ for its computation").  From kNN lists already on the device: for every (mask, query) the
 * number of listed neighbours with D <= eps_mask, their distance sum and mean, and out_complete = 1 where
 * the k-th neighbour lies beyond eps -- the list then holds the whole eps-neighbourhood and the values ARE
 * the range join's (up to the rounding of D = sqrt(d^2) against eps, the 1e-6 band of reading A2); where
 * out_complete = 0 the object still needs snaps_range_selfjoin (its count is a lower bound).
 *   knn_dist  device [n_masks][nq][k] fp32 ascending, as written by snaps_knn_selfjoin
 *   d_eps     DEVICE [n_masks] fp32 (e.g. a column of snaps_eps_search's output)
 *   out_count device [n_masks][nq] uint32; out_sumdist, out_mean fp32 or NULL; out_complete uint8 or NULL
 */
snaps_status snaps_range_from_knn(int64_t nq, int n_masks, int k, const float *knn_dist,
                                  const float *d_eps, uint32_t *out_count, float *out_sumdist,
                                  float *out_mean, uint8_t *out_complete, void *stream);

/*
 * ---- a8: batched ("oversubscribed") joins for outputs that exceed device
 * (or host) memory.  Masks are processed in groups of masks_per_batch; each group's outputs are
 * produced into a two-slot device staging ring inside d_workspace and copied on a side stream
 * to the host while the next group computes.  The workspace must hold
 * snaps_workspace_bytes(...) + snaps_stream_ring_bytes(nq, N, k, masks_per_batch).
 *
 * snaps_knn_selfjoin_streamed: the destination is the caller's full-size PINNED HOST arrays
 * (shapes of snaps_knn_selfjoin's outputs; any may be NULL, at least one non-NULL); `stream`
 * completes only after the last host copy has landed.
 */
size_t snaps_stream_ring_bytes(int64_t nq, int64_t N, int k, int masks_per_batch);

snaps_status snaps_knn_selfjoin_streamed(const float *d_X, int64_t N, int n_feat, int64_t ld,
                                         const uint16_t *h_masks, int n_masks, int k,
                                         int masks_per_batch,
                                         int64_t q_begin, int64_t q_end, int flags,
                                         int32_t *h_out_idx, float *h_out_dist,
                                         float *h_out_kth, float *h_out_mean,
                                         int32_t *h_out_indeg,
                                         void *d_workspace, size_t workspace_bytes, void *stream);

/*
 * The recycling sink: when the whole output does not fit on the host either (the kNN lists of the
 * all-subspace run are 83 GB, of the LSST-scale run 164 GB), each group is copied into one of a
 * few pinned host buffers and handed to a consumer callback, after which the buffer is reused.
 *
 *   want        which outputs to produce (SNAPS_OUT_* bits)
 *   h_buffers   n_buffers >= 2 pinned host buffers of buffer_bytes >=
 *               snaps_sink_batch_bytes(nq, N, k, masks_per_batch, want) each
 *   consume     called on the calling thread, once per group in mask order, with pointers into
 *               the buffer; the buffer is recycled when it returns
 * These two calls return after the last group has been consumed (the consumer runs on the host).
 */
#define SNAPS_OUT_IDX 1u
#define SNAPS_OUT_DIST 2u
#define SNAPS_OUT_KTH 4u
#define SNAPS_OUT_MEAN 8u
#define SNAPS_OUT_INDEG 16u
#define SNAPS_OUT_COUNT 32u
#define SNAPS_OUT_SUMDIST 64u
#define SNAPS_OUT_EPSMEAN 128u

typedef struct snaps_batch_view {
    int mask_begin, mask_end;   /* this group = masks [mask_begin, mask_end) of the caller's list */
    int64_t q_begin, q_end;     /* its queries */
    int64_t N;
    int k;
    const int32_t *idx;         /* [mask_end - mask_begin][nq][k], or NULL */
    const float *dist;
    const float *kth;           /* [..][nq] */
    const float *mean;
    const int32_t *indeg;       /* [..][N] */
    const uint32_t *count;      /* [..][nq] */
    const float *sumdist;
    const float *eps_mean;
} snaps_batch_view;

typedef void (*snaps_batch_fn)(void *user, const snaps_batch_view *view);

typedef struct snaps_batch_sink {
    void **h_buffers;
    int n_buffers;
    size_t buffer_bytes;
    unsigned want;
    snaps_batch_fn consume;
    void *user;
} snaps_batch_sink;

size_t snaps_sink_batch_bytes(int64_t nq, int64_t N, int k, int masks_per_batch, unsigned want);

snaps_status snaps_knn_selfjoin_sink(const float *d_X, int64_t N, int n_feat, int64_t ld,
                                     const uint16_t *h_masks, int n_masks, int k, int masks_per_batch,
                                     int64_t q_begin, int64_t q_end, int flags,
                                     const snaps_batch_sink *sink,
                                     void *d_workspace, size_t workspace_bytes, void *stream);

snaps_status snaps_range_selfjoin_sink(const float *d_X, int64_t N, int n_feat, int64_t ld,
                                       const uint16_t *h_masks, int n_masks, const float *h_eps,
                                       int masks_per_batch,
                                       int64_t q_begin, int64_t q_end, int flags,
                                       const snaps_batch_sink *sink,
                                       void *d_workspace, size_t workspace_bytes, void *stream);

/*
 * Peak-rate probe used for the roofline denominator:
 * runs an FP32 instruction-throughput microkernel on `stream` and returns the
 * measured warp-instruction lane rate.  kind: 0 = FFMA (two of three operands uniform), 1 = FADD,
 * 2 = FADD + FSETP pairs (the sub-lattice join's inner-loop mix), 3 = FFMA with three
 * register operands, 4 = packed FFMA2 (fma.rn.f32x2, two results per lane: counted as two
 * lane-ops), 5 = packed FADD2.  *h_lane_ops_per_s
 * receives executed lane-ops per second (one FFMA counts as ONE lane-op).
 * d_scratch: device, >= 4096 bytes.  Synchronises `stream` (it returns a measurement).
 */
snaps_status snaps_probe_fp32_rate(int kind, double *h_lane_ops_per_s, void *d_scratch, void *stream);

/*
 * ---- NEXT-1 (PAPER.md sections 3.4, 3.5.2, 3.6): ranking and parameter selection ----
 *
 * Metric kinds: which end of a score is outlying.
 */
#define SNAPS_METRIC_DSSJ_COUNT 0   /* uint32 counts, fewest neighbours = most outlying */
#define SNAPS_METRIC_DSSJ_MEAN 1    /* fp32 mean eps-distance, largest = most outlying; objects
                                       with count 0 rank first; needs d_counts */
#define SNAPS_METRIC_KNN_INDEGREE 2 /* int32 in-degree, lowest = most outlying */
#define SNAPS_METRIC_KNN_MEAN 3     /* fp32 mean (or k-th) kNN distance, largest = most outlying */

/* Device scratch snaps_rank_scores needs for n_rows score rows of N objects. */
size_t snaps_rank_workspace_bytes(int64_t N, int n_rows);

/*
 * Ranking function R (Table 2): for each of n_rows rows of N
 * scores, out_rank[row][i] = dense rank of object i, 0 = most outlying, equal scores share a
 * rank; out_order[row][p] = id of the p-th most outlying object, ties in increasing id order
 * (the "top-n" of Eq. 2 is its first n entries, reading A15).  d_values: device,
 * [n_rows][N], uint32 / fp32 / int32 per metric kind (scores are non-negative); d_counts:
 * device [n_rows][N], only for SNAPS_METRIC_DSSJ_MEAN.  Either output may be NULL.
 */
snaps_status snaps_rank_scores(int metric, const void *d_values, const uint32_t *d_counts,
                               int64_t N, int n_rows, int32_t *out_rank, int32_t *out_order,
                               void *d_workspace, size_t workspace_bytes, void *stream);

/*
 * Eq. 2: out_f[row] = |top-n(A[row]) ∩ top-n(B[row])| / n, from two
 * out_order arrays ([n_rows][N] each, device).  1 <= n <= N.
 */
snaps_status snaps_topn_overlap(const int32_t *d_order_a, const int32_t *d_order_b, int64_t N,
                                int n_rows, int n, float *out_f, void *stream);

/*
 * Eq. 3: out_j[row] = the first j in 0..G-1 that minimises
 * |U_min[j][row] - U_max[j][row]|.  d_u_min, d_u_max: device, [G][n_rows] fp32.  n_top > 0: the n
 * of Eq. 2 that made the fractions; they are taken back to integer hit counts first so that equal
 * differences compare equal (ties must not hang on rounding).  n_top = 0: compare the floats.
 */
snaps_status snaps_select_parameter(const float *d_u_min, const float *d_u_max, int G, int n_rows,
                                    int n_top, int32_t *out_j, void *stream);

/*
 * k grid: scores for k_j <= k_max from lists computed once for k_max (their
 * first k_j entries).  knn_idx/knn_dist: [n_masks][N][k_max] as written by
 * snaps_knn_selfjoin; outputs [n_masks][N], any may be NULL; out_indeg is zeroed here.
 */
snaps_status snaps_knn_scores_at_k(int64_t N, int n_masks, int k_max, int k_j,
                                   const int32_t *knn_idx, const float *knn_dist,
                                   float *out_kth, float *out_mean, int32_t *out_indeg,
                                   void *stream);

/*
 * k^select per feature space (Eq. 2 and Eq. 3 applied to the k grid): from lists
 * computed once for k_max, for every k_j of the grid derive the scores (prefix), rank them, compare
 * the top-n sets with those of the smallest and the largest k, and select the k_j that minimises
 * |U_min - U_max| -- for the distance-oblivious metric (in-degree) and the distance-aware metric
 * (mean kNN distance).
 *   knn_idx, knn_dist  device, [n_masks][N][k_max] as written by snaps_knn_selfjoin
 *   h_k_grid           host, [G] ascending, 1 <= k_j <= k_max, G >= 2
 *   n_top              n of Eq. 2 (the paper uses 0.01 |D|), 1 <= n_top <= N
 *   out_j_indeg, out_j_mean   device, [n_masks] int32: index into the grid of the selected k
 *   out_u                     device, [4][G][n_masks] fp32 or NULL: U_min / U_max of the in-degree
 *                             metric, then U_min / U_max of the mean-distance metric
 * Workspace: snaps_select_k_workspace_bytes(N, n_masks, G).
 */
size_t snaps_select_k_workspace_bytes(int64_t N, int n_masks, int G);

snaps_status snaps_knn_select_k(int64_t N, int n_masks, int k_max, const int32_t *knn_idx,
                                const float *knn_dist, const int32_t *h_k_grid, int G, int n_top,
                                int32_t *out_j_indeg, int32_t *out_j_mean, float *out_u,
                                void *d_workspace, size_t workspace_bytes, void *stream);

/*
 * DSSJ for a grid of radii in ONE scan (Fig. 3: "we execute DSSJ once for
 * eps_max and use this result set to derive the result sets for all eps_i in G").
 *   h_eps_grid  host, [n_masks][G] fp32, per mask strictly ascending, finite, > 0; 1 <= G <= 32
 *   out_count   device, [n_masks][G][nq] uint32: neighbours within eps_g (self excluded)
 *   out_sumdist, out_mean  device, same shape, fp32; may be NULL (mean = 0 when count = 0)
 *   q_begin, q_end, flags  as for snaps_range_selfjoin (both engines have a radius-grid kernel;
 *               the grid engine is the one for large selectivities such as PAPER.md:229's
 *               s_max ~ 0.15 |D|, where nearly every pair is a hit)
 * Workspace: snaps_range_grid_workspace_bytes(N, n_feat, n_masks, G, flags).
 */
size_t snaps_range_grid_workspace_bytes(int64_t N, int n_feat, int n_masks, int G, int flags);

snaps_status snaps_range_selfjoin_grid(const float *d_X, int64_t N, int n_feat, int64_t ld,
                                       const uint16_t *h_masks, int n_masks,
                                       const float *h_eps_grid, int G,
                                       int64_t q_begin, int64_t q_end, int flags,
                                       uint32_t *out_count, float *out_sumdist, float *out_mean,
                                       void *d_workspace, size_t workspace_bytes, void *stream);

/*
 * ---- NEXT-2: search radius for a target selectivity ----
 *
 * Sampled distance histogram: for every mask, out_hist[mask][b] = number of ordered pairs (q in
 * the query sample, c in the candidate sample, c != q by index) whose distance D(q, c; mask) falls
 * in bin b of n_bins equal bins over [0, h_rmax[mask]); farther pairs are not counted.
 *   h_sample_q [nq], h_sample_c [nc]  host, object ids in 0..N-1
 *   h_rmax [n_masks]                  host, > 0: the largest radius of interest per mask
 *   out_hist                          device, [n_masks][n_bins] uint64, zeroed by the call
 *   1 <= n_bins <= 8192; workspace: snaps_dist_hist_workspace_bytes(nq, nc, n_masks)
 */
size_t snaps_dist_hist_workspace_bytes(int nq, int nc, int n_masks);

snaps_status snaps_sample_distance_histogram(const float *d_X, int64_t N, int n_feat, int64_t ld,
                                             const uint16_t *h_masks, int n_masks,
                                             const int32_t *h_sample_q, int nq,
                                             const int32_t *h_sample_c, int nc, const float *h_rmax,
                                             int n_bins, unsigned long long *out_hist,
                                             void *d_workspace, size_t workspace_bytes, void *stream);

/*
 * The whole search of PAPER.md:229-237 in one call, on the device: (1) eps_mean[mask] = the mean
 * distance over the sampled (query, candidate) pairs, c != q by index -- "the upper bound on a
 * practical search radius"; (2) the histogram of those distances in n_bins equal bins
 * over [0, eps_mean); (3) for every target selectivity s_t (mean neighbours per point, PAPER.md:221;
 * the paper's eps_min / eps_max are s = 0.001 |D| and 0.15 |D|) the upper edge of the first bin whose
 * cumulative mean cum * (N-1) / pairs reaches s_t, or eps_mean if none does.
 *   h_sample_q [nq], h_sample_c [nc]  host, distinct object ids each
 *   h_target_s [n_targets]            host, > 0
 *   out_eps_mean  device [n_masks] fp32;  out_eps  device [n_masks][n_targets] fp32
 *   out_hist      device [n_masks][n_bins] uint64 or NULL (the histogram, for inspection)
 * Workspace: snaps_eps_search_workspace_bytes(nq, nc, n_masks, n_bins, n_targets).
 */
size_t snaps_eps_search_workspace_bytes(int nq, int nc, int n_masks, int n_bins, int n_targets);

snaps_status snaps_eps_search(const float *d_X, int64_t N, int n_feat, int64_t ld,
                              const uint16_t *h_masks, int n_masks,
                              const int32_t *h_sample_q, int nq, const int32_t *h_sample_c, int nc,
                              int n_bins, const double *h_target_s, int n_targets,
                              float *out_eps_mean, float *out_eps, unsigned long long *out_hist,
                              void *d_workspace, size_t workspace_bytes, void *stream);

/*
 * eps^select per feature space in one call (section 3.5.2, 229-239 section 3.5.3) --
 * the DSSJ twin of snaps_knn_select_k: (1) eps_min and eps_max for the selectivities s_min < s_max by
 * snaps_eps_search; (2) the grid of G evenly spaced radii between them (fp32; |G| is not given in the
 * paper, reading A17); (3) one range join at eps_max binned over the grid; (4) for
 * the neighbour-count metric and the mean-distance metric: ranks at every radius, their top-n overlap
 * with the ranks at eps_min (U_min) and at eps_max (U_max) (Eq. 2), and the radius that minimises
 * |U_min - U_max| (Eq. 3).
 *   out_eps_grid   device [n_masks][G] fp32 or NULL: the radii
 *   out_j_count, out_j_mean  device [n_masks] int32: index of the selected radius per metric
 *   out_u          device [4][G][n_masks] fp32 or NULL (as snaps_knn_select_k)
 * Workspace: snaps_select_eps_workspace_bytes(...) (it holds the [n_masks][G][N] scores and orders:
 * call it on a few hundred masks at a time).
 */
size_t snaps_select_eps_workspace_bytes(int64_t N, int n_feat, int n_masks, int G, int nq, int nc,
                                        int n_bins, int flags);

snaps_status snaps_range_select_eps(const float *d_X, int64_t N, int n_feat, int64_t ld,
                                    const uint16_t *h_masks, int n_masks,
                                    const int32_t *h_sample_q, int nq, const int32_t *h_sample_c, int nc,
                                    int n_bins, double s_min, double s_max, int G, int n_top, int flags,
                                    float *out_eps_grid, int32_t *out_j_count, int32_t *out_j_mean,
                                    float *out_u, void *d_workspace, size_t workspace_bytes, void *stream);

/*
 * Host arithmetic on a histogram copied back from the device: the cumulative histogram gives the
 * mean number of neighbours per point at each bin edge, mean(r_b) = cum[b] * (N-1) / (nq * nc')
 * with nc' = candidates per query (nc, minus one where the query is in the candidate sample --
 * passed as pairs_per_mask = total ordered pairs examined); h_eps[mask] = the smallest bin edge
 * whose mean reaches target_s, or h_rmax[mask] if none does.
 */
snaps_status snaps_eps_from_histogram(const unsigned long long *h_hist, int n_masks, int n_bins,
                                      const float *h_rmax, int64_t N, int64_t pairs_per_mask,
                                      double target_s, float *h_eps);

/*
 * Kernel timing for roofline reports.  While enabled
 * (per calling thread), every join call records a CUDA event pair on `stream`
 * around each launch of its dominant (join) kernel; the pairs of the most
 * recent call of this thread are kept.
 * snaps_profile_last_kernel_ms synchronises on them and returns the summed
 * device time in milliseconds and the number of launches (either pointer may
 * be NULL).  Disabled by default; enabling costs two event records per launch.
 */
snaps_status snaps_profile_enable(int on);
snaps_status snaps_profile_last_kernel_ms(float *h_ms, int *h_launches);

#ifdef __cplusplus
}
#endif
#endif /* SNAPS_H */
