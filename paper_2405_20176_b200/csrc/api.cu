// api.cu -- C ABI of libsnaps (include/snaps.h): argument checks, the host-side mask-batch
// planner (step a2), workspace carving, kernel launches and the pinned-host output ring (a8).
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <utility>
#include <vector>

#include "../../include/snaps.h"
#include "knn_lattice.cuh"
#include "misc_kernels.cuh"
#include "pivot_sort.cuh"
#include "eps_search.cuh"
#include "range_grid.cuh"
#include "range_lattice.cuh"
#include "ranking.cuh"

namespace {

thread_local char g_err[512] = "";

snaps_status fail(snaps_status code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                      \
    do {                                                                                    \
        cudaError_t e_ = (expr);                                                            \
        if (e_ != cudaSuccess)                                                              \
            return fail(SNAPS_CUDA_ERROR, "%s: %s (%s:%d)", #expr, cudaGetErrorString(e_),  \
                        __FILE__, __LINE__);                                                \
    } while (0)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ---- optional event pairs around the join kernels (snaps_profile_*) ----
bool g_prof_on = false;
std::vector<std::pair<cudaEvent_t, cudaEvent_t>> g_prof_pool;  // created once, reused
size_t g_prof_used = 0;

void prof_reset() { g_prof_used = 0; }

bool prof_begin(cudaStream_t st) {
    if (!g_prof_on) return false;
    if (g_prof_used == g_prof_pool.size()) {
        cudaEvent_t a, b;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return false;
        g_prof_pool.emplace_back(a, b);
    }
    cudaEventRecord(g_prof_pool[g_prof_used].first, st);
    return true;
}

void prof_end(bool began, cudaStream_t st) {
    if (!began) return;
    cudaEventRecord(g_prof_pool[g_prof_used].second, st);
    ++g_prof_used;
}

int n_tiles_for(int64_t N) { return static_cast<int>((N + snaps::kTileRows - 1) / snaps::kTileRows); }

// Gray rank of the 9 high-feature bits: consecutive batches differ in one feature, which is
// what makes the previous batch's neighbours good threshold seeds.
uint32_t gray_rank(uint32_t gray) {
    uint32_t b = gray;
    for (uint32_t s = 1; s < 16; s <<= 1) b ^= b >> s;
    return b;
}

// Step a2.  One batch per distinct set H of features 6..14; slot[T] = position of mask H|T.
// A mask listed more than once gets a further batch with the same H.
void plan_lattice(const uint16_t* masks, int n_masks, const float* thr,
                  std::vector<snaps::BatchDesc>* out) {
    std::map<uint32_t, std::vector<int>> by_h;  // gray rank of H -> batch indices
    std::vector<snaps::BatchDesc>& B = *out;
    B.clear();
    for (int m = 0; m < n_masks; ++m) {
        const uint32_t H = masks[m] & ~static_cast<uint32_t>(snaps::kLat - 1);
        const int T = masks[m] & (snaps::kLat - 1);
        std::vector<int>& lst = by_h[gray_rank(H >> snaps::kLow)];
        int use = -1;
        for (int bi : lst)
            if (B[bi].slot[T] < 0) {
                use = bi;
                break;
            }
        if (use < 0) {
            snaps::BatchDesc d;
            d.hmask = H;
            d.n_valid = 0;
            d.pivot = (H >> snaps::kLow) ? snaps::kLow + __builtin_ctz(H >> snaps::kLow) : -1;
            d.pad_ = 0;
            for (int t = 0; t < snaps::kLat; ++t) {
                d.slot[t] = -1;
                d.thr[t] = -1.f;
            }
            B.push_back(d);
            use = static_cast<int>(B.size()) - 1;
            lst.push_back(use);
        }
        B[use].slot[T] = m;
        B[use].n_valid += 1;
        if (thr) B[use].thr[T] = thr[m];
    }
    std::vector<snaps::BatchDesc> ordered;
    ordered.reserve(B.size());
    for (auto& kv : by_h)
        for (int bi : kv.second) ordered.push_back(B[bi]);
    B.swap(ordered);
}

// Pivot sweep only: a batch without high features has no pivot and would take a full pass.  Split
// it by lattice feature instead -- the masks that contain feature 0, then of the rest those that
// contain feature 1, ... -- so that every piece has a feature all its masks share (its pivot).
void split_for_sweep(std::vector<snaps::BatchDesc>* batches) {
    std::vector<snaps::BatchDesc> out;
    for (const snaps::BatchDesc& b : *batches) {
        if (b.pivot >= 0) {
            out.push_back(b);
            continue;
        }
        bool taken[snaps::kLat] = {false};
        for (int f = 0; f < snaps::kLow; ++f) {
            snaps::BatchDesc d = b;
            d.n_valid = 0;
            d.pivot = f;
            for (int t = 0; t < snaps::kLat; ++t) {
                const bool mine = b.slot[t] >= 0 && !taken[t] && ((t >> f) & 1);
                if (mine) {
                    taken[t] = true;
                    d.n_valid += 1;
                } else {
                    d.slot[t] = -1;
                    d.thr[t] = -1.f;
                }
            }
            if (d.n_valid > 0) out.push_back(d);
        }
    }
    batches->swap(out);
}

snaps_status check_common(const float* d_X, int64_t N, int n_feat, int64_t ld,
                          const uint16_t* h_masks, int n_masks) {
    if (!d_X) return fail(SNAPS_INVALID_ARG, "d_X is NULL");
    if (reinterpret_cast<uintptr_t>(d_X) % 4 != 0) return fail(SNAPS_INVALID_ARG, "d_X not 4-byte aligned");
    if (N < 2) return fail(SNAPS_INVALID_ARG, "N = %lld < 2", (long long)N);
    if (N > (int64_t)1 << 30) return fail(SNAPS_UNSUPPORTED, "N = %lld > 2^30", (long long)N);
    if (n_feat < 1 || n_feat > SNAPS_MAX_FEATURES)
        return fail(SNAPS_INVALID_ARG, "n_feat = %d outside 1..15", n_feat);
    if (ld < n_feat) return fail(SNAPS_INVALID_ARG, "ld = %lld < n_feat", (long long)ld);
    if (!h_masks || n_masks < 1) return fail(SNAPS_INVALID_ARG, "no masks");
    for (int m = 0; m < n_masks; ++m) {
        if (h_masks[m] == 0) return fail(SNAPS_INVALID_ARG, "mask %d is zero", m);
        if ((h_masks[m] >> n_feat) != 0)
            return fail(SNAPS_INVALID_ARG, "mask %d (0x%x) has a bit >= n_feat", m, h_masks[m]);
    }
    return SNAPS_OK;
}

// Large tables take the pivot sweep (pivot_sort.cuh); SNAPS_KNN_SWEEP=0/1 overrides the size rule.
bool use_sweep(int64_t N) {
    if (const char* e = getenv("SNAPS_KNN_SWEEP")) return atoi(e) != 0;
    return N >= (1 << 18);
}

struct Workspace {
    unsigned char* pivot;   // 9 pivot sets + sort scratch (only when use_sweep(N))
    float* Xp;
    float4* Xb;
    int* counter;
    snaps::BatchDesc* batches;
    unsigned char* ring;   // rest
    size_t ring_bytes;
};

int n_blocks_for(int64_t N) { return static_cast<int>((N + 31) / 32); }



// one pivot set: sorted blocked table, sorted values, position -> id, id -> position
size_t pivot_set_bytes(int64_t N) {
    const size_t n_pad = static_cast<size_t>(n_blocks_for(N)) * 32;
    return align_up(n_pad * 64, 256) + 2 * align_up(n_pad * 4, 256) + align_up(static_cast<size_t>(N) * 4, 256);
}

size_t pivot_region_bytes(int64_t N) {
    return 15 * pivot_set_bytes(N) + align_up(snaps::pivot_sort_temp_bytes(n_blocks_for(N) * 32), 256);
}

size_t base_workspace_bytes(int64_t N, int n_masks, int k) {
    const size_t table = align_up(static_cast<size_t>(n_tiles_for(N)) * snaps::kTileBytes, 256);
    const size_t blocked = align_up(static_cast<size_t>(n_blocks_for(N)) * 2048, 256);
    const size_t batches = align_up(static_cast<size_t>(n_masks) * sizeof(snaps::BatchDesc), 256);
    const size_t pivot = use_sweep(N) ? pivot_region_bytes(N) : 0;
    return table + blocked + 256 + batches + pivot;
}

snaps_status carve(void* d_ws, size_t bytes, int64_t N, int n_masks, int k, Workspace* w) {
    if (!d_ws) return fail(SNAPS_INVALID_ARG, "d_workspace is NULL");
    if (reinterpret_cast<uintptr_t>(d_ws) % 256 != 0)
        return fail(SNAPS_INVALID_ARG, "d_workspace not 256-byte aligned");
    const size_t need = base_workspace_bytes(N, n_masks, k);
    if (bytes < need)
        return fail(SNAPS_WORKSPACE_TOO_SMALL, "workspace %zu < %zu bytes", bytes, need);
    unsigned char* p = static_cast<unsigned char*>(d_ws);
    const size_t table = align_up(static_cast<size_t>(n_tiles_for(N)) * snaps::kTileBytes, 256);
    const size_t blocked = align_up(static_cast<size_t>(n_blocks_for(N)) * 2048, 256);
    const size_t batches = align_up(static_cast<size_t>(n_masks) * sizeof(snaps::BatchDesc), 256);
    w->Xp = reinterpret_cast<float*>(p);
    w->Xb = reinterpret_cast<float4*>(p + table);
    w->counter = reinterpret_cast<int*>(p + table + blocked);
    w->batches = reinterpret_cast<snaps::BatchDesc*>(p + table + blocked + 256);
    w->pivot = p + table + blocked + 256 + batches;
    w->ring = p + need;
    w->ring_bytes = bytes - need;
    return SNAPS_OK;
}

// Pointers of pivot set j (feature j) inside the pivot region.
struct PivotSet {
    float4* Xs;
    float* piv;
    int* idmap;
    int* pos;
};

PivotSet pivot_set(const Workspace& w, int64_t N, int j) {
    const size_t n_pad = static_cast<size_t>(n_blocks_for(N)) * 32;
    unsigned char* b = w.pivot + static_cast<size_t>(j) * pivot_set_bytes(N);
    PivotSet s;
    s.Xs = reinterpret_cast<float4*>(b);
    s.piv = reinterpret_cast<float*>(b + align_up(n_pad * 64, 256));
    s.idmap = reinterpret_cast<int*>(b + align_up(n_pad * 64, 256) + align_up(n_pad * 4, 256));
    s.pos = reinterpret_cast<int*>(b + align_up(n_pad * 64, 256) + 2 * align_up(n_pad * 4, 256));
    return s;
}

// Build the sorted copies for the pivot features the batches use (lowest high feature of each).
snaps_status build_pivots(const Workspace& w, int64_t N, const std::vector<snaps::BatchDesc>& batches,
                          cudaStream_t st) {
    bool need[15] = {false};
    for (const snaps::BatchDesc& b : batches)
        if (b.pivot >= 0) need[b.pivot] = true;
    const int n_pad = n_blocks_for(N) * 32;
    void* temp = w.pivot + 15 * pivot_set_bytes(N);
    const size_t temp_bytes = snaps::pivot_sort_temp_bytes(n_pad);
    for (int j = 0; j < 15; ++j) {
        if (!need[j]) continue;
        const PivotSet s = pivot_set(w, N, j);
        CUDA_TRY(snaps::pivot_build(w.Xp, static_cast<int>(N), n_pad, j, s.Xs, s.piv, s.idmap,
                                    s.pos, temp, temp_bytes, st));
    }
    return SNAPS_OK;
}

int sm_count() {
    static int cached = 0;
    if (!cached) {
        int dev = 0, n = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0)
            cached = n;
        else
            cached = 148;
    }
    return cached;
}

int knn_warps_for(int k) {
    // per-warp list state in shared memory; what is left of the 256 KB array stays L1 for the
    // table stream
    const size_t budget = 227 * 1024;
    int w = snaps::kKnnMaxThreads / 32;
    if (const char* e = getenv("SNAPS_KNN_WARPS")) {   // tuning knob: warps (queries) per CTA
        const int v = atoi(e);
        if (v >= 1 && v <= snaps::kKnnMaxThreads / 32 && snaps::knn_lattice_smem_bytes(k, v) <= 227 * 1024) return v;
    }
    while (w > 1 && snaps::knn_lattice_smem_bytes(k, w) > budget) --w;
    return w;
}

// Launch the kNN kernel over descriptors already uploaded at d_batches[0..nb).
snaps_status knn_enqueue(const Workspace& w, const snaps::BatchDesc* d_batches, int nb, int64_t N, int k,
                         int32_t* out_idx, float* out_dist, float* out_kth, float* out_mean,
                         int32_t* out_indeg, cudaStream_t st) {
    CUDA_TRY(cudaMemsetAsync(w.counter, 0, 256, st));
    snaps::KnnParams p;
    p.Xp = w.Xp;
    p.Xb = w.Xb;
    p.n_blocks = n_blocks_for(N);
    p.sweep = use_sweep(N) ? 1 : 0;
    for (int j = 0; j < 15; ++j) {
        const PivotSet s = p.sweep ? pivot_set(w, N, j) : PivotSet{nullptr, nullptr, nullptr, nullptr};
        p.Xs[j] = s.Xs;
        p.piv[j] = s.piv;
        p.idmap[j] = s.idmap;
        p.pos[j] = s.pos;
    }
    p.N = static_cast<int>(N);
    p.k = k;
    p.batches = d_batches;
    p.n_batches = nb;
    p.warps = knn_warps_for(k);
    // runs of 8 consecutive batches: long enough for the previous batch's neighbours to seed the
    // next one, short enough that the in-degree rows of the batches in flight (8 x 64 x 4N bytes)
    // stay in L2; items are plentiful (N per run), so the per-warp scheduler balances the tail
    int run = 8;
    if (const char* e = getenv("SNAPS_KNN_RUN")) {      // tuning knob: batches per work item
        const int v = atoi(e);
        if (v >= 1) run = v;
    }
    p.batches_per_item = std::min(nb, run);
    p.n_bchunks = (nb + p.batches_per_item - 1) / p.batches_per_item;
    p.work_counter = reinterpret_cast<unsigned long long*>(w.counter);
    p.out_idx = out_idx;
    p.out_dist = out_dist;
    p.out_kth = out_kth;
    p.out_mean = out_mean;
    p.out_indeg = out_indeg;
    const int64_t items = N * p.n_bchunks;
    const int grid = static_cast<int>(std::min<int64_t>((items + p.warps - 1) / p.warps, sm_count()));
    const bool prof = prof_begin(st);
    CUDA_TRY(snaps::knn_lattice_launch(p, grid, st));
    prof_end(prof, st);
    return SNAPS_OK;
}

}  // namespace

extern "C" {

const char* snaps_last_error(void) { return g_err; }

const char* snaps_version(void) { return "snaps-b200 0.1 (sm_100a)"; }

size_t snaps_workspace_bytes(int64_t N, int n_feat, int n_masks, int k) {
    if (N < 2 || n_feat < 1 || n_feat > SNAPS_MAX_FEATURES || n_masks < 1 || k < 0 || k > SNAPS_MAX_K)
        return 0;
    return base_workspace_bytes(N, n_masks, k);
}

int64_t snaps_planned_evals(int64_t N, int n_feat, const uint16_t* h_masks, int n_masks) {
    if (!h_masks || n_masks < 1 || N < 2 || n_feat < 1 || n_feat > SNAPS_MAX_FEATURES) return -1;
    std::vector<snaps::BatchDesc> b;
    plan_lattice(h_masks, n_masks, nullptr, &b);
    return static_cast<int64_t>(b.size()) * snaps::kLat * N * N;
}

snaps_status snaps_knn_selfjoin(const float* d_X, int64_t N, int n_feat, int64_t ld,
                                const uint16_t* h_masks, int n_masks, int k, int32_t* out_idx,
                                float* out_dist, float* out_kth, float* out_mean,
                                int32_t* out_indeg, void* d_workspace, size_t workspace_bytes,
                                void* stream) {
    prof_reset();
    snaps_status rc = check_common(d_X, N, n_feat, ld, h_masks, n_masks);
    if (rc) return rc;
    if (k < 1 || k > SNAPS_MAX_K || k > N - 1)
        return fail(SNAPS_INVALID_ARG, "k = %d outside 1..min(N-1, %d)", k, SNAPS_MAX_K);
    if (!out_idx && !out_dist && !out_kth && !out_mean && !out_indeg)
        return fail(SNAPS_INVALID_ARG, "all outputs are NULL");
    Workspace w;
    rc = carve(d_workspace, workspace_bytes, N, n_masks, k, &w);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    std::vector<snaps::BatchDesc> batches;
    plan_lattice(h_masks, n_masks, nullptr, &batches);
    const int n_tiles = n_tiles_for(N);
    CUDA_TRY(snaps::stage_table_launch(d_X, ld, static_cast<int>(N), n_feat, w.Xp,
                                       n_tiles * snaps::kTileRows, st));
    CUDA_TRY(snaps::stage_blocked_launch(d_X, ld, static_cast<int>(N), n_feat, w.Xb, n_blocks_for(N), st));
    if (use_sweep(N)) {
        split_for_sweep(&batches);
        rc = build_pivots(w, N, batches, st);
        if (rc) return rc;
    }
    if (out_indeg)
        CUDA_TRY(cudaMemsetAsync(out_indeg, 0, sizeof(int32_t) * static_cast<size_t>(n_masks) * N, st));
    CUDA_TRY(cudaMemcpyAsync(w.batches, batches.data(), sizeof(snaps::BatchDesc) * batches.size(),
                             cudaMemcpyHostToDevice, st));
    return knn_enqueue(w, w.batches, static_cast<int>(batches.size()), N, k, out_idx, out_dist, out_kth,
                       out_mean, out_indeg, st);
}

snaps_status snaps_range_selfjoin(const float* d_X, int64_t N, int n_feat, int64_t ld,
                                  const uint16_t* h_masks, int n_masks, const float* h_eps,
                                  uint32_t* out_count, float* out_sumdist, float* out_mean,
                                  void* d_workspace, size_t workspace_bytes, void* stream) {
    prof_reset();
    snaps_status rc = check_common(d_X, N, n_feat, ld, h_masks, n_masks);
    if (rc) return rc;
    if (!h_eps) return fail(SNAPS_INVALID_ARG, "h_eps is NULL");
    if (!out_count) return fail(SNAPS_INVALID_ARG, "out_count is NULL");
    std::vector<float> thr(n_masks);
    for (int m = 0; m < n_masks; ++m) {
        if (!(h_eps[m] > 0.f) || !isfinite(h_eps[m]))
            return fail(SNAPS_INVALID_ARG, "eps[%d] = %g is not finite and > 0", m, (double)h_eps[m]);
        // D <= eps  <=>  D^2 <= eps^2: compare d^2 < nextafter(fl(eps^2)) (closed ball, reading A2)
        const float e2 = static_cast<float>(static_cast<double>(h_eps[m]) * static_cast<double>(h_eps[m]));
        thr[m] = nextafterf(e2, INFINITY);
    }
    Workspace w;
    rc = carve(d_workspace, workspace_bytes, N, n_masks, 1, &w);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    std::vector<snaps::BatchDesc> batches;
    plan_lattice(h_masks, n_masks, thr.data(), &batches);
    if (use_sweep(N)) split_for_sweep(&batches);
    const int nb = static_cast<int>(batches.size());
    const int n_tiles = n_tiles_for(N);
    CUDA_TRY(snaps::stage_table_launch(d_X, ld, static_cast<int>(N), n_feat, w.Xp,
                                       n_tiles * snaps::kTileRows, st));
    CUDA_TRY(cudaMemcpyAsync(w.batches, batches.data(), sizeof(snaps::BatchDesc) * nb,
                             cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemsetAsync(w.counter, 0, 256, st));
    CUDA_TRY(snaps::stage_blocked_launch(d_X, ld, static_cast<int>(N), n_feat, w.Xb, n_blocks_for(N), st));
    if (use_sweep(N)) {
        rc = build_pivots(w, N, batches, st);
        if (rc) return rc;
    }
    snaps::RangeParams p;
    p.Xp = w.Xp;
    p.Xb = w.Xb;
    p.n_blocks = n_blocks_for(N);
    p.sweep = use_sweep(N) ? 1 : 0;
    for (int j = 0; j < 15; ++j) {
        const PivotSet s = p.sweep ? pivot_set(w, N, j) : PivotSet{nullptr, nullptr, nullptr, nullptr};
        p.Xs[j] = s.Xs;
        p.piv[j] = s.piv;
        p.idmap[j] = s.idmap;
        p.pos[j] = s.pos;
    }
    p.N = static_cast<int>(N);
    p.batches = w.batches;
    p.n_batches = nb;
    p.warps = snaps::kRangeMaxThreads / 32;
    p.batches_per_item = std::min(nb, 8);
    p.n_bchunks = (nb + p.batches_per_item - 1) / p.batches_per_item;
    p.work_counter = reinterpret_cast<unsigned long long*>(w.counter);
    p.out_count = out_count;
    p.out_sum = out_sumdist;
    p.out_mean = out_mean;
    const int64_t items = N * p.n_bchunks;
    const int grid = static_cast<int>(std::min<int64_t>((items + p.warps - 1) / p.warps, sm_count()));
    const bool prof = prof_begin(st);
    CUDA_TRY(snaps::range_lattice_launch(p, grid, st));
    prof_end(prof, st);
    return SNAPS_OK;
}

snaps_status snaps_outlier_scores(int64_t N, int n_masks, int k, const int32_t* knn_idx,
                                  const float* knn_dist, const uint32_t* eps_count,
                                  const float* eps_sumdist, float* out_kth, float* out_knn_mean,
                                  int32_t* out_indegree, float* out_eps_mean, void* stream) {
    if (N < 2 || n_masks < 1) return fail(SNAPS_INVALID_ARG, "bad sizes");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const bool want_knn = out_kth || out_knn_mean || out_indegree;
    if (want_knn) {
        if (k < 1 || k > SNAPS_MAX_K) return fail(SNAPS_INVALID_ARG, "k = %d outside 1..%d", k, SNAPS_MAX_K);
        if ((out_kth || out_knn_mean) && !knn_dist) return fail(SNAPS_INVALID_ARG, "knn_dist is NULL");
        if (out_indegree && !knn_idx) return fail(SNAPS_INVALID_ARG, "knn_idx is NULL");
        if (out_indegree)
            CUDA_TRY(cudaMemsetAsync(out_indegree, 0, sizeof(int32_t) * static_cast<size_t>(n_masks) * N, st));
        CUDA_TRY(snaps::knn_scores_launch(N, n_masks, k, knn_idx, knn_dist, out_kth, out_knn_mean,
                                          out_indegree, st));
    }
    if (out_eps_mean) {
        if (!eps_count || !eps_sumdist) return fail(SNAPS_INVALID_ARG, "eps inputs are NULL");
        CUDA_TRY(snaps::eps_mean_launch(N * n_masks, eps_count, eps_sumdist, out_eps_mean, st));
    }
    if (!want_knn && !out_eps_mean) return fail(SNAPS_INVALID_ARG, "all outputs are NULL");
    return SNAPS_OK;
}

size_t snaps_stream_ring_bytes(int64_t N, int k, int masks_per_batch) {
    if (N < 2 || k < 1 || masks_per_batch < 1) return 0;
    // two staging slots, each: idx + dist lists and three score arrays for one mask group
    const size_t per_mask = align_up(static_cast<size_t>(N) * (2 * static_cast<size_t>(k) + 3) * 4, 256) + 5 * 256;
    return 2 * per_mask * static_cast<size_t>(masks_per_batch);
}

snaps_status snaps_knn_selfjoin_streamed(const float* d_X, int64_t N, int n_feat, int64_t ld,
                                         const uint16_t* h_masks, int n_masks, int k,
                                         int masks_per_batch, int32_t* h_out_idx, float* h_out_dist,
                                         float* h_out_kth, float* h_out_mean, int32_t* h_out_indeg,
                                         void* d_workspace, size_t workspace_bytes, void* stream) {
    prof_reset();
    snaps_status rc = check_common(d_X, N, n_feat, ld, h_masks, n_masks);
    if (rc) return rc;
    if (k < 1 || k > SNAPS_MAX_K || k > N - 1)
        return fail(SNAPS_INVALID_ARG, "k = %d outside 1..min(N-1, %d)", k, SNAPS_MAX_K);
    if (masks_per_batch < 1) return fail(SNAPS_INVALID_ARG, "masks_per_batch < 1");
    if (!h_out_idx && !h_out_dist && !h_out_kth && !h_out_mean && !h_out_indeg)
        return fail(SNAPS_INVALID_ARG, "all outputs are NULL");
    Workspace w;
    rc = carve(d_workspace, workspace_bytes, N, n_masks, k, &w);
    if (rc) return rc;
    const size_t ring_need = snaps_stream_ring_bytes(N, k, masks_per_batch);
    if (w.ring_bytes < ring_need)
        return fail(SNAPS_WORKSPACE_TOO_SMALL, "workspace ring %zu < %zu bytes", w.ring_bytes, ring_need);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int n_tiles = n_tiles_for(N);
    CUDA_TRY(snaps::stage_table_launch(d_X, ld, static_cast<int>(N), n_feat, w.Xp,
                                       n_tiles * snaps::kTileRows, st));
    CUDA_TRY(snaps::stage_blocked_launch(d_X, ld, static_cast<int>(N), n_feat, w.Xb, n_blocks_for(N), st));

    const size_t mpb = static_cast<size_t>(masks_per_batch);
    const size_t n_list = align_up(mpb * N * k * 4, 256);
    const size_t n_score = align_up(mpb * N * 4, 256);
    struct Slot {
        int32_t* idx;
        float* dist;
        float* kth;
        float* mean;
        int32_t* indeg;
    } slots[2];
    unsigned char* r = w.ring;
    for (int s = 0; s < 2; ++s) {
        slots[s].idx = reinterpret_cast<int32_t*>(r); r += n_list;
        slots[s].dist = reinterpret_cast<float*>(r); r += n_list;
        slots[s].kth = reinterpret_cast<float*>(r); r += n_score;
        slots[s].mean = reinterpret_cast<float*>(r); r += n_score;
        slots[s].indeg = reinterpret_cast<int32_t*>(r); r += n_score;
    }
    // Plan every mask group up front and upload all descriptors with one copy, so that the
    // loop below only enqueues (no host<->device synchronisation between groups).
    std::vector<snaps::BatchDesc> all_batches;
    std::vector<size_t> group_off;
    for (int m0 = 0; m0 < n_masks; m0 += masks_per_batch) {
        std::vector<snaps::BatchDesc> b;
        plan_lattice(h_masks + m0, std::min(masks_per_batch, n_masks - m0), nullptr, &b);
        if (use_sweep(N)) split_for_sweep(&b);
        group_off.push_back(all_batches.size());
        all_batches.insert(all_batches.end(), b.begin(), b.end());
    }
    group_off.push_back(all_batches.size());
    if (use_sweep(N)) {
        rc = build_pivots(w, N, all_batches, st);
        if (rc) return rc;
    }
    CUDA_TRY(cudaMemcpyAsync(w.batches, all_batches.data(), sizeof(snaps::BatchDesc) * all_batches.size(),
                             cudaMemcpyHostToDevice, st));
    cudaStream_t side;
    CUDA_TRY(cudaStreamCreateWithFlags(&side, cudaStreamNonBlocking));
    cudaEvent_t computed[2], copied[2];
    for (int s = 0; s < 2; ++s) {
        CUDA_TRY(cudaEventCreateWithFlags(&computed[s], cudaEventDisableTiming));
        CUDA_TRY(cudaEventCreateWithFlags(&copied[s], cudaEventDisableTiming));
    }
    snaps_status result = SNAPS_OK;
    int group = 0;
    for (int m0 = 0; m0 < n_masks && result == SNAPS_OK; m0 += masks_per_batch, ++group) {
        const int nm = std::min(masks_per_batch, n_masks - m0);
        const int s = group & 1;
        if (group >= 2) {
            // staging slot s is free once its previous copy-out has finished
            cudaError_t e = cudaStreamWaitEvent(st, copied[s], 0);
            if (e != cudaSuccess) { result = fail(SNAPS_CUDA_ERROR, "cudaStreamWaitEvent: %s", cudaGetErrorString(e)); break; }
        }
        if (h_out_indeg) {
            cudaError_t e = cudaMemsetAsync(slots[s].indeg, 0, sizeof(int32_t) * static_cast<size_t>(nm) * N, st);
            if (e != cudaSuccess) { result = fail(SNAPS_CUDA_ERROR, "cudaMemsetAsync: %s", cudaGetErrorString(e)); break; }
        }
        result = knn_enqueue(w, w.batches + group_off[group],
                             static_cast<int>(group_off[group + 1] - group_off[group]), N, k,
                             h_out_idx ? slots[s].idx : nullptr,
                             h_out_dist ? slots[s].dist : nullptr, h_out_kth ? slots[s].kth : nullptr,
                             h_out_mean ? slots[s].mean : nullptr, h_out_indeg ? slots[s].indeg : nullptr, st);
        if (result != SNAPS_OK) break;
        cudaEventRecord(computed[s], st);
        cudaStreamWaitEvent(side, computed[s], 0);
        const size_t off_list = static_cast<size_t>(m0) * N * k, off_score = static_cast<size_t>(m0) * N;
        const size_t b_list = static_cast<size_t>(nm) * N * k * 4, b_score = static_cast<size_t>(nm) * N * 4;
        cudaError_t e = cudaSuccess;
        if (h_out_idx && e == cudaSuccess) e = cudaMemcpyAsync(h_out_idx + off_list, slots[s].idx, b_list, cudaMemcpyDeviceToHost, side);
        if (h_out_dist && e == cudaSuccess) e = cudaMemcpyAsync(h_out_dist + off_list, slots[s].dist, b_list, cudaMemcpyDeviceToHost, side);
        if (h_out_kth && e == cudaSuccess) e = cudaMemcpyAsync(h_out_kth + off_score, slots[s].kth, b_score, cudaMemcpyDeviceToHost, side);
        if (h_out_mean && e == cudaSuccess) e = cudaMemcpyAsync(h_out_mean + off_score, slots[s].mean, b_score, cudaMemcpyDeviceToHost, side);
        if (h_out_indeg && e == cudaSuccess) e = cudaMemcpyAsync(h_out_indeg + off_score, slots[s].indeg, b_score, cudaMemcpyDeviceToHost, side);
        if (e != cudaSuccess) { result = fail(SNAPS_CUDA_ERROR, "cudaMemcpyAsync D2H: %s", cudaGetErrorString(e)); break; }
        cudaEventRecord(copied[s], side);
    }
    // the caller's stream completes only after the last copies have landed
    for (int s = 0; s < 2 && s < group; ++s) cudaStreamWaitEvent(st, copied[s], 0);
    for (int s = 0; s < 2; ++s) {
        cudaEventDestroy(computed[s]);
        cudaEventDestroy(copied[s]);
    }
    cudaStreamDestroy(side);
    return result;
}

size_t snaps_range_grid_workspace_bytes(int64_t N, int n_feat, int n_masks, int G) {
    if (N < 2 || n_feat < 1 || n_feat > SNAPS_MAX_FEATURES || n_masks < 1 || G < 1 || G > snaps::kRangeGridMaxRadii)
        return 0;
    return base_workspace_bytes(N, n_masks, 0) + align_up(static_cast<size_t>(n_masks) * G * 4, 256);
}

snaps_status snaps_range_selfjoin_grid(const float* d_X, int64_t N, int n_feat, int64_t ld,
                                       const uint16_t* h_masks, int n_masks, const float* h_eps_grid, int G,
                                       uint32_t* out_count, float* out_sumdist, float* out_mean,
                                       void* d_workspace, size_t workspace_bytes, void* stream) {
    prof_reset();
    snaps_status rc = check_common(d_X, N, n_feat, ld, h_masks, n_masks);
    if (rc) return rc;
    if (!h_eps_grid || !out_count) return fail(SNAPS_INVALID_ARG, "NULL eps grid or out_count");
    if (G < 1 || G > snaps::kRangeGridMaxRadii) return fail(SNAPS_INVALID_ARG, "G = %d outside 1..%d", G, snaps::kRangeGridMaxRadii);
    std::vector<float> thr(static_cast<size_t>(n_masks) * G);
    for (int m = 0; m < n_masks; ++m)
        for (int g = 0; g < G; ++g) {
            const float e = h_eps_grid[static_cast<size_t>(m) * G + g];
            if (!(e > 0.f) || !isfinite(e) || (g > 0 && !(e > h_eps_grid[static_cast<size_t>(m) * G + g - 1])))
                return fail(SNAPS_INVALID_ARG, "eps_grid[%d][%d] = %g: radii must be finite, > 0 and ascending", m, g, (double)e);
            const float e2 = static_cast<float>(static_cast<double>(e) * static_cast<double>(e));
            thr[static_cast<size_t>(m) * G + g] = nextafterf(e2, INFINITY);   // closed ball, reading A2
        }
    Workspace w;
    rc = carve(d_workspace, workspace_bytes, N, n_masks, 0, &w);
    if (rc) return rc;
    const size_t grid_bytes = align_up(static_cast<size_t>(n_masks) * G * 4, 256);
    if (w.ring_bytes < grid_bytes)
        return fail(SNAPS_WORKSPACE_TOO_SMALL, "workspace lacks %zu bytes for the radius grid", grid_bytes);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    std::vector<snaps::BatchDesc> batches;
    plan_lattice(h_masks, n_masks, nullptr, &batches);
    const int nb = static_cast<int>(batches.size());
    CUDA_TRY(snaps::stage_table_launch(d_X, ld, static_cast<int>(N), n_feat, w.Xp,
                                       n_tiles_for(N) * snaps::kTileRows, st));
    CUDA_TRY(snaps::stage_blocked_launch(d_X, ld, static_cast<int>(N), n_feat, w.Xb, n_blocks_for(N), st));
    CUDA_TRY(cudaMemcpyAsync(w.batches, batches.data(), sizeof(snaps::BatchDesc) * nb, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(w.ring, thr.data(), thr.size() * 4, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaStreamSynchronize(st));   // thr is a host temporary: the copy must land before it goes away
    CUDA_TRY(cudaMemsetAsync(w.counter, 0, 256, st));
    snaps::RangeGridParams p;
    p.Xp = w.Xp;
    p.Xb = w.Xb;
    p.n_blocks = n_blocks_for(N);
    p.N = static_cast<int>(N);
    p.G = G;
    p.batches = w.batches;
    p.n_batches = nb;
    p.thr_grid = reinterpret_cast<const float*>(w.ring);
    p.warps = snaps::kRangeGridMaxThreads / 32;
    while (p.warps > 1 && snaps::range_grid_smem_bytes(G, p.warps) > 227 * 1024) --p.warps;
    p.work_counter = reinterpret_cast<unsigned long long*>(w.counter);
    p.out_count = out_count;
    p.out_sum = out_sumdist;
    p.out_mean = out_mean;
    const int64_t items = N * nb;
    const int grid = static_cast<int>(std::min<int64_t>((items + p.warps - 1) / p.warps, sm_count()));
    const bool prof = prof_begin(st);
    CUDA_TRY(snaps::range_grid_launch(p, grid, st));
    prof_end(prof, st);
    return SNAPS_OK;
}

size_t snaps_dist_hist_workspace_bytes(int nq, int nc, int n_masks) {
    if (nq < 1 || nc < 1 || n_masks < 1) return 0;
    return snaps::dist_hist_workspace_bytes(nq, nc, n_masks);
}

snaps_status snaps_sample_distance_histogram(const float* d_X, int64_t N, int n_feat, int64_t ld,
                                             const uint16_t* h_masks, int n_masks, const int32_t* h_sample_q,
                                             int nq, const int32_t* h_sample_c, int nc, const float* h_rmax,
                                             int n_bins, unsigned long long* out_hist, void* d_workspace,
                                             size_t workspace_bytes, void* stream) {
    snaps_status rc = check_common(d_X, N, n_feat, ld, h_masks, n_masks);
    if (rc) return rc;
    if (!h_sample_q || !h_sample_c || !h_rmax || !out_hist || nq < 1 || nc < 1)
        return fail(SNAPS_INVALID_ARG, "NULL or empty samples");
    if (n_bins < 1 || n_bins > 8192) return fail(SNAPS_INVALID_ARG, "n_bins = %d outside 1..8192", n_bins);
    for (int i = 0; i < nq; ++i)
        if (h_sample_q[i] < 0 || h_sample_q[i] >= N) return fail(SNAPS_INVALID_ARG, "query sample id out of range");
    for (int i = 0; i < nc; ++i)
        if (h_sample_c[i] < 0 || h_sample_c[i] >= N) return fail(SNAPS_INVALID_ARG, "candidate sample id out of range");
    for (int m = 0; m < n_masks; ++m)
        if (!(h_rmax[m] > 0.f) || !isfinite(h_rmax[m])) return fail(SNAPS_INVALID_ARG, "rmax[%d] not finite and > 0", m);
    if (!d_workspace || workspace_bytes < snaps::dist_hist_workspace_bytes(nq, nc, n_masks))
        return fail(SNAPS_WORKSPACE_TOO_SMALL, "histogram workspace too small");
    CUDA_TRY(snaps::dist_hist_launch(d_X, ld, n_feat, h_sample_q, nq, h_sample_c, nc, h_masks, h_rmax, n_masks,
                                     n_bins, out_hist, d_workspace, static_cast<cudaStream_t>(stream)));
    return SNAPS_OK;
}

snaps_status snaps_eps_from_histogram(const unsigned long long* h_hist, int n_masks, int n_bins, const float* h_rmax,
                                      int64_t N, int64_t pairs_per_mask, double target_s, float* h_eps) {
    if (!h_hist || !h_rmax || !h_eps || n_masks < 1 || n_bins < 1 || N < 2 || pairs_per_mask < 1 || !(target_s > 0.0))
        return fail(SNAPS_INVALID_ARG, "bad arguments");
    for (int m = 0; m < n_masks; ++m) {
        unsigned long long cum = 0;
        h_eps[m] = h_rmax[m];
        for (int b = 0; b < n_bins; ++b) {
            cum += h_hist[static_cast<size_t>(m) * n_bins + b];
            const double mean = static_cast<double>(cum) * static_cast<double>(N - 1) / static_cast<double>(pairs_per_mask);
            if (mean >= target_s) {
                h_eps[m] = static_cast<float>(static_cast<double>(h_rmax[m]) * (b + 1) / n_bins);
                break;
            }
        }
    }
    return SNAPS_OK;
}

size_t snaps_select_k_workspace_bytes(int64_t N, int n_masks) {
    if (N < 2 || n_masks < 1) return 0;
    const size_t arr = align_up(static_cast<size_t>(N) * n_masks * 4, 256);
    // score array, three order arrays (smallest k, largest k, current k), ranking scratch
    return 4 * arr + align_up(snaps::rank_workspace_bytes(N, n_masks), 256);
}

snaps_status snaps_knn_select_k(int64_t N, int n_masks, int k_max, const int32_t* knn_idx, const float* knn_dist,
                                const int32_t* h_k_grid, int G, int n_top, int32_t* out_j_indeg,
                                int32_t* out_j_mean, float* out_u, void* d_workspace, size_t workspace_bytes,
                                void* stream) {
    if (N < 2 || n_masks < 1 || k_max < 1 || !knn_idx || !knn_dist || !h_k_grid)
        return fail(SNAPS_INVALID_ARG, "bad sizes or NULL inputs");
    if (G < 2 || G > 256) return fail(SNAPS_INVALID_ARG, "G = %d outside 2..256", G);
    for (int j = 0; j < G; ++j)
        if (h_k_grid[j] < 1 || h_k_grid[j] > k_max || (j > 0 && h_k_grid[j] <= h_k_grid[j - 1]))
            return fail(SNAPS_INVALID_ARG, "k grid must ascend within 1..k_max (entry %d = %d)", j, h_k_grid[j]);
    if (n_top < 1 || n_top > N) return fail(SNAPS_INVALID_ARG, "n_top = %d outside 1..N", n_top);
    if (!out_j_indeg || !out_j_mean) return fail(SNAPS_INVALID_ARG, "NULL outputs");
    if ((N + 31) / 32 * 4 > 200 * 1024) return fail(SNAPS_UNSUPPORTED, "N too large for the top-n bitmap");
    if (!d_workspace || workspace_bytes < snaps_select_k_workspace_bytes(N, n_masks))
        return fail(SNAPS_WORKSPACE_TOO_SMALL, "workspace %zu < %zu bytes", workspace_bytes,
                    snaps_select_k_workspace_bytes(N, n_masks));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t arr = align_up(static_cast<size_t>(N) * n_masks * 4, 256);
    unsigned char* p = static_cast<unsigned char*>(d_workspace);
    void* score = p;
    int32_t* ord_min = reinterpret_cast<int32_t*>(p + arr);
    int32_t* ord_max = reinterpret_cast<int32_t*>(p + 2 * arr);
    int32_t* ord_cur = reinterpret_cast<int32_t*>(p + 3 * arr);
    void* rws = p + 4 * arr;
    const size_t rws_bytes = workspace_bytes - 4 * arr;
    float* u_tmp = nullptr;   // U arrays live in out_u if given, else in a temporary device buffer
    float* u = out_u;
    if (!u) {
        CUDA_TRY(cudaMallocAsync(&u_tmp, sizeof(float) * 4 * G * static_cast<size_t>(n_masks), st));
        u = u_tmp;
    }
    snaps_status rc = SNAPS_OK;
    for (int metric = 0; metric < 2 && rc == SNAPS_OK; ++metric) {
        const int kind = metric == 0 ? SNAPS_METRIC_KNN_INDEGREE : SNAPS_METRIC_KNN_MEAN;
        float* u_min = u + static_cast<size_t>(2 * metric) * G * n_masks;
        float* u_max = u + static_cast<size_t>(2 * metric + 1) * G * n_masks;
        auto order_for = [&](int kj, int32_t* ord) -> cudaError_t {
            cudaError_t e;
            if (metric == 0) {
                e = cudaMemsetAsync(score, 0, sizeof(int32_t) * static_cast<size_t>(n_masks) * N, st);
                if (e != cudaSuccess) return e;
                e = snaps::scores_at_k_launch(N, n_masks, k_max, kj, knn_idx, nullptr, nullptr, nullptr,
                                              static_cast<int32_t*>(score), st);
            } else {
                e = snaps::scores_at_k_launch(N, n_masks, k_max, kj, nullptr, knn_dist, nullptr,
                                              static_cast<float*>(score), nullptr, st);
            }
            if (e != cudaSuccess) return e;
            return snaps::rank_launch(kind, score, nullptr, N, n_masks, nullptr, ord, rws, rws_bytes, st);
        };
        cudaError_t e = order_for(h_k_grid[0], ord_min);
        if (e == cudaSuccess) e = order_for(h_k_grid[G - 1], ord_max);
        for (int j = 0; j < G && e == cudaSuccess; ++j) {
            const int32_t* oc = j == 0 ? ord_min : (j == G - 1 ? ord_max : ord_cur);
            if (j > 0 && j < G - 1) e = order_for(h_k_grid[j], ord_cur);
            if (e == cudaSuccess)
                e = snaps::topn_overlap_launch(ord_min, oc, N, n_masks, n_top, u_min + static_cast<size_t>(j) * n_masks, st);
            if (e == cudaSuccess)
                e = snaps::topn_overlap_launch(ord_max, oc, N, n_masks, n_top, u_max + static_cast<size_t>(j) * n_masks, st);
        }
        if (e == cudaSuccess)
            e = snaps::select_launch(u_min, u_max, G, n_masks, n_top, metric == 0 ? out_j_indeg : out_j_mean, st);
        if (e != cudaSuccess) rc = fail(SNAPS_CUDA_ERROR, "select_k: %s", cudaGetErrorString(e));
    }
    if (u_tmp) cudaFreeAsync(u_tmp, st);
    return rc;
}

size_t snaps_rank_workspace_bytes(int64_t N, int n_rows) {
    if (N < 1 || n_rows < 1) return 0;
    return snaps::rank_workspace_bytes(N, n_rows);
}

snaps_status snaps_rank_scores(int metric, const void* d_values, const uint32_t* d_counts, int64_t N,
                               int n_rows, int32_t* out_rank, int32_t* out_order, void* d_workspace,
                               size_t workspace_bytes, void* stream) {
    if (metric < 0 || metric > 3) return fail(SNAPS_INVALID_ARG, "metric kind %d outside 0..3", metric);
    if (!d_values || N < 1 || n_rows < 1) return fail(SNAPS_INVALID_ARG, "bad sizes or NULL values");
    if (N > (int64_t)1 << 30) return fail(SNAPS_UNSUPPORTED, "N = %lld > 2^30", (long long)N);
    if (metric == SNAPS_METRIC_DSSJ_MEAN && !d_counts) return fail(SNAPS_INVALID_ARG, "d_counts is NULL");
    if (!out_rank && !out_order) return fail(SNAPS_INVALID_ARG, "all outputs are NULL");
    if (!d_workspace || workspace_bytes < snaps::rank_workspace_bytes(N, n_rows))
        return fail(SNAPS_WORKSPACE_TOO_SMALL, "rank workspace %zu < %zu bytes", workspace_bytes,
                    snaps::rank_workspace_bytes(N, n_rows));
    CUDA_TRY(snaps::rank_launch(metric, d_values, d_counts, N, n_rows, out_rank, out_order, d_workspace,
                                workspace_bytes, static_cast<cudaStream_t>(stream)));
    return SNAPS_OK;
}

snaps_status snaps_topn_overlap(const int32_t* d_order_a, const int32_t* d_order_b, int64_t N, int n_rows,
                                int n, float* out_f, void* stream) {
    if (!d_order_a || !d_order_b || !out_f) return fail(SNAPS_INVALID_ARG, "NULL argument");
    if (N < 1 || n_rows < 1 || n < 1 || n > N) return fail(SNAPS_INVALID_ARG, "bad sizes (n = %d, N = %lld)", n, (long long)N);
    if ((N + 31) / 32 * 4 > 200 * 1024) return fail(SNAPS_UNSUPPORTED, "N = %lld: bitmap exceeds shared memory", (long long)N);
    CUDA_TRY(snaps::topn_overlap_launch(d_order_a, d_order_b, N, n_rows, n, out_f, static_cast<cudaStream_t>(stream)));
    return SNAPS_OK;
}

snaps_status snaps_select_parameter(const float* d_u_min, const float* d_u_max, int G, int n_rows, int n_top,
                                    int32_t* out_j, void* stream) {
    if (!d_u_min || !d_u_max || !out_j || G < 1 || n_rows < 1 || n_top < 0) return fail(SNAPS_INVALID_ARG, "bad arguments");
    CUDA_TRY(snaps::select_launch(d_u_min, d_u_max, G, n_rows, n_top, out_j, static_cast<cudaStream_t>(stream)));
    return SNAPS_OK;
}

snaps_status snaps_knn_scores_at_k(int64_t N, int n_masks, int k_max, int k_j, const int32_t* knn_idx,
                                   const float* knn_dist, float* out_kth, float* out_mean,
                                   int32_t* out_indeg, void* stream) {
    if (N < 2 || n_masks < 1 || k_max < 1 || k_j < 1 || k_j > k_max) return fail(SNAPS_INVALID_ARG, "bad sizes");
    if ((out_kth || out_mean) && !knn_dist) return fail(SNAPS_INVALID_ARG, "knn_dist is NULL");
    if (out_indeg && !knn_idx) return fail(SNAPS_INVALID_ARG, "knn_idx is NULL");
    if (!out_kth && !out_mean && !out_indeg) return fail(SNAPS_INVALID_ARG, "all outputs are NULL");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (out_indeg) CUDA_TRY(cudaMemsetAsync(out_indeg, 0, sizeof(int32_t) * static_cast<size_t>(n_masks) * N, st));
    CUDA_TRY(snaps::scores_at_k_launch(N, n_masks, k_max, k_j, knn_idx, knn_dist, out_kth, out_mean, out_indeg, st));
    return SNAPS_OK;
}

snaps_status snaps_profile_enable(int on) {
    g_prof_on = on != 0;
    prof_reset();
    return SNAPS_OK;
}

snaps_status snaps_profile_last_kernel_ms(float* h_ms, int* h_launches) {
    float total = 0.f;
    for (size_t i = 0; i < g_prof_used; ++i) {
        CUDA_TRY(cudaEventSynchronize(g_prof_pool[i].second));
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, g_prof_pool[i].first, g_prof_pool[i].second));
        total += ms;
    }
    if (h_ms) *h_ms = total;
    if (h_launches) *h_launches = static_cast<int>(g_prof_used);
    return SNAPS_OK;
}

snaps_status snaps_probe_fp32_rate(int kind, double* h_lane_ops_per_s, void* stream) {
    if (kind < 0 || kind > 2 || !h_lane_ops_per_s) return fail(SNAPS_INVALID_ARG, "bad probe arguments");
    double ops = 0.0;
    float ms = 0.f;
    CUDA_TRY(snaps::probe_fp32_launch(kind, &ops, &ms, static_cast<cudaStream_t>(stream)));
    *h_lane_ops_per_s = ops / (static_cast<double>(ms) * 1e-3);
    return SNAPS_OK;
}

}  // extern "C"
