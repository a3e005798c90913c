// api.cu -- C ABI of libsnaps (include/snaps.h): argument checks, the host-side mask-batch
// planner (step a2), engine selection, workspace carving, kernel launches and the batched
// output paths (a8: staging ring, side-stream D2H, pinned-host destinations or a recycling sink).
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <iterator>
#include <map>
#include <utility>
#include <mutex>
#include <vector>

#include "../../include/snaps.h"
#include "eps_search.cuh"
#include "grid_index.cuh"
#include "grid_join.cuh"
#include "knn_bigk.cuh"
#include "knn_lattice.cuh"
#include "misc_kernels.cuh"
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

// ---- optional event pairs around the join kernels (snaps_profile_*), per calling thread ----
struct Prof {
    bool on = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> pool;  // created once, reused
    size_t used = 0;
};
thread_local Prof g_prof;

void prof_reset() { g_prof.used = 0; }

bool prof_begin(cudaStream_t st) {
    if (!g_prof.on) return false;
    if (g_prof.used == g_prof.pool.size()) {
        cudaEvent_t a, b;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return false;
        g_prof.pool.emplace_back(a, b);
    }
    cudaEventRecord(g_prof.pool[g_prof.used].first, st);
    return true;
}

void prof_end(bool began, cudaStream_t st) {
    if (!began) return;
    cudaEventRecord(g_prof.pool[g_prof.used].second, st);
    ++g_prof.used;
}

// ---- side stream and events of the batched calls, per calling thread, created on first use ----
struct Side {
    cudaStream_t stream = nullptr;
    cudaEvent_t computed[2] = {nullptr, nullptr}, copied[2] = {nullptr, nullptr};
};
thread_local Side g_side;

cudaError_t side_get(Side** out) {
    if (!g_side.stream) {
        cudaError_t e = cudaStreamCreateWithFlags(&g_side.stream, cudaStreamNonBlocking);
        for (int s = 0; s < 2 && e == cudaSuccess; ++s) {
            e = cudaEventCreateWithFlags(&g_side.computed[s], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&g_side.copied[s], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) return e;
    }
    *out = &g_side;
    return cudaSuccess;
}

int n_tiles_for(int64_t N) { return static_cast<int>((N + snaps::kTileRows - 1) / snaps::kTileRows); }
int n_blocks_for(int64_t N) { return static_cast<int>((N + 31) / 32); }

// Gray rank of the 9 high-feature bits: consecutive batches differ in one feature, which is
// what makes the previous batch's neighbours good threshold seeds.
uint32_t gray_rank(uint32_t gray) {
    uint32_t b = gray;
    for (uint32_t s = 1; s < 16; s <<= 1) b ^= b >> s;
    return b;
}

// Step a2.  One batch per distinct set H of features 6..14; slot[T] = position of mask H|T
// (+ slot_base).  A mask listed more than once gets a further batch with the same H.
void plan_lattice(const uint16_t* masks, int n_masks, const float* thr, int slot_base,
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
            d.pad_[0] = d.pad_[1] = 0;
            for (int t = 0; t < snaps::kLat; ++t) {
                d.slot[t] = -1;
                d.thr[t] = -1.f;
            }
            B.push_back(d);
            use = static_cast<int>(B.size()) - 1;
            lst.push_back(use);
        }
        B[use].slot[T] = slot_base + m;
        B[use].n_valid += 1;
        if (thr) B[use].thr[T] = thr[m];
    }
    std::vector<snaps::BatchDesc> ordered;
    ordered.reserve(B.size());
    for (auto& kv : by_h)
        for (int bi : kv.second) ordered.push_back(B[bi]);
    B.swap(ordered);
}

int popcount16(uint32_t m) { return __builtin_popcount(m & 0xffffu); }

// ---- what every join call shares ---------------------------------------------------------
struct Job {
    const float* X;          // caller's table (device, or host with SNAPS_FLAG_X_ON_HOST)
    int64_t N;
    int n_feat;
    int64_t ld;
    const uint16_t* h_masks;
    int n_masks;
    int64_t q_begin, q_end;
    int flags;
    int engine;
    int64_t nq() const { return q_end - q_begin; }
};

int resolve_engine(int flags, int64_t N, int k) {
    const int e = flags & SNAPS_ENGINE_MASK;
    if (e != SNAPS_ENGINE_AUTO) return e;
    return (N >= (1 << 18) || k > SNAPS_LATTICE_MAX_K) ? SNAPS_ENGINE_GRID : SNAPS_ENGINE_LATTICE;
}

snaps_status check_job(const Job& j, int k_for_engine) {
    if (!j.X) return fail(SNAPS_INVALID_ARG, "X is NULL");
    if (reinterpret_cast<uintptr_t>(j.X) % 4 != 0) return fail(SNAPS_INVALID_ARG, "X not 4-byte aligned");
    if (j.N < 2) return fail(SNAPS_INVALID_ARG, "N = %lld < 2", (long long)j.N);
    if (j.N > (int64_t)1 << 30) return fail(SNAPS_UNSUPPORTED, "N = %lld > 2^30", (long long)j.N);
    if (j.n_feat < 1 || j.n_feat > SNAPS_MAX_FEATURES)
        return fail(SNAPS_INVALID_ARG, "n_feat = %d outside 1..15", j.n_feat);
    if (j.ld < j.n_feat) return fail(SNAPS_INVALID_ARG, "ld = %lld < n_feat", (long long)j.ld);
    if (!j.h_masks || j.n_masks < 1) return fail(SNAPS_INVALID_ARG, "no masks");
    for (int m = 0; m < j.n_masks; ++m) {
        if (j.h_masks[m] == 0) return fail(SNAPS_INVALID_ARG, "mask %d is zero", m);
        if ((j.h_masks[m] >> j.n_feat) != 0)
            return fail(SNAPS_INVALID_ARG, "mask %d (0x%x) has a bit >= n_feat", m, j.h_masks[m]);
    }
    if (j.q_begin < 0 || j.q_end > j.N || j.q_begin >= j.q_end)
        return fail(SNAPS_INVALID_ARG, "query range [%lld, %lld) not within [0, N)", (long long)j.q_begin,
                    (long long)j.q_end);
    if (j.flags & ~(SNAPS_ENGINE_MASK | SNAPS_FLAG_X_ON_HOST)) return fail(SNAPS_INVALID_ARG, "unknown flag bits 0x%x", j.flags);
    if (j.engine != SNAPS_ENGINE_LATTICE && j.engine != SNAPS_ENGINE_GRID)
        return fail(SNAPS_INVALID_ARG, "unknown engine %d", j.engine);
    if (j.engine == SNAPS_ENGINE_LATTICE && k_for_engine > SNAPS_LATTICE_MAX_K)
        return fail(SNAPS_INVALID_ARG, "k = %d: the sub-lattice engine holds k <= %d", k_for_engine, SNAPS_LATTICE_MAX_K);
    return SNAPS_OK;
}

// ---- workspace ---------------------------------------------------------------------------
// common:   [host-X copy] | Xp | counter(256)
// lattice:  Xb | batch descriptors (n_masks)
// grid:     device masks | plans | table region | index region
// then:     whatever the caller added (staging ring, radius grid)
struct Workspace {
    float* Xdense;             // dense copy of a host X, else nullptr
    float* Xp;
    unsigned long long* counter;
    float4* Xb;
    snaps::BatchDesc* batches;
    uint16_t* d_masks;
    snaps::GridPlan* plans;
    unsigned char* grid_table;
    unsigned char* grid_index;
    size_t grid_index_bytes;
    unsigned char* extra;
    size_t extra_bytes;
};

size_t base_workspace_bytes(int64_t N, int n_feat, int n_masks, int engine, int flags) {
    size_t b = 0;
    if (flags & SNAPS_FLAG_X_ON_HOST) b += align_up(static_cast<size_t>(N) * n_feat * 4, 256);
    b += align_up(static_cast<size_t>(n_tiles_for(N)) * snaps::kTileBytes, 256) + 256;
    if (engine == SNAPS_ENGINE_LATTICE) {
        b += align_up(static_cast<size_t>(n_blocks_for(N)) * 2048, 256);
        b += align_up(static_cast<size_t>(n_masks) * sizeof(snaps::BatchDesc), 256);
    } else {
        b += align_up(static_cast<size_t>(n_masks) * 2, 256);
        b += align_up(static_cast<size_t>(n_masks) * sizeof(snaps::GridPlan), 256);
        b += snaps::grid_table_bytes(N) + snaps::grid_index_bytes(N);
    }
    return b;
}

snaps_status carve(void* d_ws, size_t bytes, const Job& j, Workspace* w) {
    if (!d_ws) return fail(SNAPS_INVALID_ARG, "d_workspace is NULL");
    if (reinterpret_cast<uintptr_t>(d_ws) % 256 != 0)
        return fail(SNAPS_INVALID_ARG, "d_workspace not 256-byte aligned");
    const size_t need = base_workspace_bytes(j.N, j.n_feat, j.n_masks, j.engine, j.flags);
    if (bytes < need) return fail(SNAPS_WORKSPACE_TOO_SMALL, "workspace %zu < %zu bytes", bytes, need);
    unsigned char* p = static_cast<unsigned char*>(d_ws);
    memset(w, 0, sizeof(*w));
    if (j.flags & SNAPS_FLAG_X_ON_HOST) {
        w->Xdense = reinterpret_cast<float*>(p);
        p += align_up(static_cast<size_t>(j.N) * j.n_feat * 4, 256);
    }
    w->Xp = reinterpret_cast<float*>(p);
    p += align_up(static_cast<size_t>(n_tiles_for(j.N)) * snaps::kTileBytes, 256);
    w->counter = reinterpret_cast<unsigned long long*>(p);
    p += 256;
    if (j.engine == SNAPS_ENGINE_LATTICE) {
        w->Xb = reinterpret_cast<float4*>(p);
        p += align_up(static_cast<size_t>(n_blocks_for(j.N)) * 2048, 256);
        w->batches = reinterpret_cast<snaps::BatchDesc*>(p);
        p += align_up(static_cast<size_t>(j.n_masks) * sizeof(snaps::BatchDesc), 256);
    } else {
        w->d_masks = reinterpret_cast<uint16_t*>(p);
        p += align_up(static_cast<size_t>(j.n_masks) * 2, 256);
        w->plans = reinterpret_cast<snaps::GridPlan*>(p);
        p += align_up(static_cast<size_t>(j.n_masks) * sizeof(snaps::GridPlan), 256);
        w->grid_table = p;
        p += snaps::grid_table_bytes(j.N);
        w->grid_index = p;
        w->grid_index_bytes = snaps::grid_index_bytes(j.N);
        p += w->grid_index_bytes;
    }
    w->extra = p;
    w->extra_bytes = bytes - need;
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
    // per-warp list state in shared memory: as many warps (queries) per CTA as fit the 227 KB
    int w = snaps::kKnnMaxThreads / 32;
    while (w > 1 && snaps::knn_lattice_smem_bytes(k, w) > 227 * 1024) --w;
    return w;
}

// ---- a1 and the engine's table-level state -----------------------------------------------
struct Engine {
    Job job;
    Workspace w;
    cudaStream_t st;
    unsigned char* bigk = nullptr;   // what is left of the workspace for the long-list kNN path (knn_bigk.cu), if any
    size_t bigk_bytes = 0;
    snaps::GridTable gt;
    snaps::GridIndex gi;
};

snaps_status engine_begin(Engine* E) {
    const Job& j = E->job;
    Workspace& w = E->w;
    const float* Xdev = j.X;
    int64_t ld = j.ld;
    if (j.flags & SNAPS_FLAG_X_ON_HOST) {
        CUDA_TRY(cudaMemcpy2DAsync(w.Xdense, static_cast<size_t>(j.n_feat) * 4, j.X, static_cast<size_t>(j.ld) * 4,
                                   static_cast<size_t>(j.n_feat) * 4, static_cast<size_t>(j.N), cudaMemcpyHostToDevice,
                                   E->st));
        Xdev = w.Xdense;
        ld = j.n_feat;
    }
    CUDA_TRY(snaps::stage_table_launch(Xdev, ld, static_cast<int>(j.N), j.n_feat, w.Xp,
                                       n_tiles_for(j.N) * snaps::kTileRows, E->st));
    if (j.engine == SNAPS_ENGINE_LATTICE) {
        CUDA_TRY(snaps::stage_blocked_launch(Xdev, ld, static_cast<int>(j.N), j.n_feat, w.Xb, n_blocks_for(j.N), E->st));
    } else {
        CUDA_TRY(snaps::grid_table_build(w.Xp, static_cast<int>(j.N), j.n_feat, &E->gt, w.grid_table, w.grid_index,
                                         w.grid_index_bytes, E->st));
        snaps::grid_index_carve(w.grid_index, w.grid_index_bytes, j.N, &E->gi);
        CUDA_TRY(cudaMemcpyAsync(w.d_masks, j.h_masks, static_cast<size_t>(j.n_masks) * 2, cudaMemcpyHostToDevice, E->st));
        CUDA_TRY(snaps::grid_plan_launch(w.d_masks, j.n_masks, j.N, E->gt, w.plans, E->st));
    }
    return SNAPS_OK;
}

// The outputs of one launch group: pointers to the group's first mask row.
struct KnnOut {
    int32_t* idx;
    float* dist;
    float* kth;
    float* mean;
    int32_t* indeg;
};
struct RangeOut {
    uint32_t* count;
    float* sum;
    float* mean;
};

// ---- sub-lattice engine launches (descriptors already on the device) -----------------------
snaps_status lattice_knn_enqueue(Engine* E, const snaps::BatchDesc* d_batches, int nb, int k, const KnnOut& o) {
    const Job& j = E->job;
    CUDA_TRY(cudaMemsetAsync(E->w.counter, 0, 256, E->st));
    snaps::KnnParams p;
    p.Xp = E->w.Xp;
    p.Xb = E->w.Xb;
    p.n_blocks = n_blocks_for(j.N);
    p.N = static_cast<int>(j.N);
    p.q_begin = static_cast<int>(j.q_begin);
    p.nq = static_cast<int>(j.nq());
    p.k = k;
    p.batches = d_batches;
    p.n_batches = nb;
    p.warps = knn_warps_for(k);
    // runs of 4 consecutive batches: long enough for the previous batch's neighbours to seed the
    // next one, short enough that the in-degree rows of the batches in flight (4 x 64 x 4N bytes =
    // 32 MB at N = 31,693) stay in one half of the L2 (measured: DRAM writes = 1.03x the output with
    // runs of 4, 10x with runs of 8, same time); items are plentiful (nq per run), so the per-warp
    // scheduler balances the tail
    p.batches_per_item = std::min(nb, 4);
    p.n_bchunks = (nb + p.batches_per_item - 1) / p.batches_per_item;
    p.work_counter = E->w.counter;
    p.out_idx = o.idx;
    p.out_dist = o.dist;
    p.out_kth = o.kth;
    p.out_mean = o.mean;
    p.out_indeg = o.indeg;
    const int64_t items = j.nq() * p.n_bchunks;
    const int grid = static_cast<int>(std::min<int64_t>((items + p.warps - 1) / p.warps, sm_count()));
    const bool prof = prof_begin(E->st);
    CUDA_TRY(snaps::knn_lattice_launch(p, grid, E->st));
    prof_end(prof, E->st);
    return SNAPS_OK;
}

snaps_status lattice_range_enqueue(Engine* E, const snaps::BatchDesc* d_batches, int nb, const RangeOut& o) {
    const Job& j = E->job;
    CUDA_TRY(cudaMemsetAsync(E->w.counter, 0, 256, E->st));
    snaps::RangeParams p;
    p.Xp = E->w.Xp;
    p.Xb = E->w.Xb;
    p.n_blocks = n_blocks_for(j.N);
    p.N = static_cast<int>(j.N);
    p.q_begin = static_cast<int>(j.q_begin);
    p.nq = static_cast<int>(j.nq());
    p.batches = d_batches;
    p.n_batches = nb;
    p.warps = snaps::kRangeMaxThreads / 32;
    p.batches_per_item = std::min(nb, 8);
    p.n_bchunks = (nb + p.batches_per_item - 1) / p.batches_per_item;
    p.work_counter = E->w.counter;
    p.out_count = o.count;
    p.out_sum = o.sum;
    p.out_mean = o.mean;
    const int64_t items = j.nq() * p.n_bchunks;
    const int grid = static_cast<int>(std::min<int64_t>((items + p.warps - 1) / p.warps, sm_count()));
    const bool prof = prof_begin(E->st);
    CUDA_TRY(snaps::range_lattice_launch(p, grid, E->st));
    prof_end(prof, E->st);
    return SNAPS_OK;
}

// ---- grid engine launches: masks [m0, m0 + nm) of the job, one index + one join each --------
void grid_params_common(Engine* E, int m, snaps::GridJoinParams* p, int* d_out) {
    const Job& j = E->job;
    const int d = popcount16(j.h_masks[m]);
    memset(p, 0, sizeof(*p));
    snaps::grid_bits_for(j.N, d, p->bits);
    p->Xp = E->w.Xp;
    p->Xs = E->gi.Xs;
    p->keys = E->gi.keys;
    p->perm = E->gi.perm;
    p->cell_start = E->gi.cell_start;
    p->qlist = (j.q_begin > 0 || j.q_end < j.N) ? E->gi.qlist : nullptr;
    p->edges = E->gt.edges;
    p->plan = E->w.plans + m;
    p->N = static_cast<int>(j.N);
    p->nq = static_cast<int>(j.nq());
    p->q_begin = static_cast<int>(j.q_begin);
    *d_out = d;
}

snaps_status grid_knn_enqueue(Engine* E, int m0, int nm, int k, const KnnOut& o) {
    const Job& j = E->job;
    const size_t nq = static_cast<size_t>(j.nq()), N = static_cast<size_t>(j.N);
    for (int m = m0; m < m0 + nm; ++m) {
        snaps::GridJoinParams p;
        int d = 0;
        grid_params_common(E, m, &p, &d);
        // long lists on a small table: radix selection over brute-force passes instead of per-query heaps, when the
        // workspace has the room (snaps_workspace_bytes asks for it)
        const bool bigk = snaps::knn_bigk_pays(j.N, k) && E->bigk &&
                          E->bigk_bytes >= snaps::knn_bigk_scratch_bytes(j.nq(), k);
        CUDA_TRY(snaps::grid_index_build(E->gt, p.plan, p.N, d, p.bits, j.q_begin, j.q_end, bigk ? 0 : k, &E->gi, E->st));
        p.warp_order = E->gi.warp_order;
        const size_t r = static_cast<size_t>(m - m0);
        p.k = k;
        p.out_idx = o.idx ? o.idx + r * nq * k : nullptr;
        p.out_dist = o.dist ? o.dist + r * nq * k : nullptr;
        p.out_kth = o.kth ? o.kth + r * nq : nullptr;
        p.out_mean = o.mean ? o.mean + r * nq : nullptr;
        p.out_indeg = o.indeg ? o.indeg + r * N : nullptr;
        const bool prof = prof_begin(E->st);
        if (bigk) CUDA_TRY(snaps::knn_bigk_launch(p, d, E->bigk, E->bigk_bytes, E->st));
        else CUDA_TRY(snaps::grid_knn_launch(p, d, E->st));
        prof_end(prof, E->st);
    }
    return SNAPS_OK;
}

// G > 0: d_radii = device [n_masks][G] fl(eps^2) rows; G = 0: h_eps2 gives one value per mask
snaps_status grid_range_enqueue(Engine* E, int m0, int nm, const float* h_eps2, int G, const float* d_radii,
                                const RangeOut& o) {
    const Job& j = E->job;
    const size_t nq = static_cast<size_t>(j.nq());
    const size_t per_mask = nq * static_cast<size_t>(G > 0 ? G : 1);
    for (int m = m0; m < m0 + nm; ++m) {
        snaps::GridJoinParams p;
        int d = 0;
        grid_params_common(E, m, &p, &d);
        CUDA_TRY(snaps::grid_index_build(E->gt, p.plan, p.N, d, p.bits, j.q_begin, j.q_end, 0, &E->gi, E->st));
        const size_t r = static_cast<size_t>(m - m0);
        p.G = G;
        if (G > 0) p.eps2_grid = d_radii + static_cast<size_t>(m) * G;
        else p.eps2 = h_eps2[m];
        p.out_count = o.count + r * per_mask;
        p.out_sum = o.sum ? o.sum + r * per_mask : nullptr;
        p.out_rmean = o.mean ? o.mean + r * per_mask : nullptr;
        const bool prof = prof_begin(E->st);
        CUDA_TRY(snaps::grid_range_launch(p, d, E->st));
        prof_end(prof, E->st);
    }
    return SNAPS_OK;
}

// fl(eps^2) and nextafter(fl(eps^2)): D <= eps <=> d^2 <= fl(eps^2) <=> d^2 < nextafter (closed ball, reading A2)
snaps_status eps_squares(const float* h_eps, size_t n, std::vector<float>* e2, std::vector<float>* thr) {
    e2->resize(n);
    thr->resize(n);
    for (size_t m = 0; m < n; ++m) {
        if (!(h_eps[m] > 0.f) || !isfinite(h_eps[m]))
            return fail(SNAPS_INVALID_ARG, "eps[%zu] = %g is not finite and > 0", m, (double)h_eps[m]);
        (*e2)[m] = static_cast<float>(static_cast<double>(h_eps[m]) * static_cast<double>(h_eps[m]));
        (*thr)[m] = nextafterf((*e2)[m], INFINITY);
    }
    return SNAPS_OK;
}

// ---- a8: mask groups -> staging ring -> side-stream D2H -> host destination -----------------
// One output array of a group: bytes per mask, device staging pointer (per slot), host destination.
struct OutArray {
    size_t bytes_per_mask;
    unsigned char* stage[2];
    unsigned char* h_full;      // streamed call: the caller's full-size array (offset by mask), or
    size_t sink_offset;         // sink call: offset inside the recycled host buffer
    bool want;
};

struct Batched {
    Engine* E;
    int k;                       // 0 = range join
    const float* h_eps2;         // range join (grid engine)
    int masks_per_batch;
    OutArray arr[5];             // knn: idx, dist, kth, mean, indeg; range: count, sum, mean
    int n_arr;
    const snaps_batch_sink* sink;   // nullptr = full-size pinned arrays
};

size_t ring_bytes(int64_t nq, int64_t N, int k, int mpb) {
    // two staging slots, each: two list arrays, two score arrays and the in-degree rows (kNN); the range
    // join's count, sum and mean fit the same space
    const size_t m = static_cast<size_t>(mpb);
    const size_t slot = 2 * align_up(static_cast<size_t>(nq) * k * 4 * m, 256) + 2 * align_up(static_cast<size_t>(nq) * 4 * m, 256) +
                        align_up(static_cast<size_t>(N) * 4 * m, 256);
    return 2 * slot;
}

snaps_status run_batched(Batched* B, const std::vector<snaps::BatchDesc>* all_batches, const std::vector<size_t>* group_off) {
    Engine* E = B->E;
    const Job& j = E->job;
    Side* side = nullptr;
    CUDA_TRY(side_get(&side));
    // carve the staging ring
    unsigned char* r = E->w.extra;
    size_t left = E->w.extra_bytes;
    for (int s = 0; s < 2; ++s)
        for (int a = 0; a < B->n_arr; ++a) {
            const size_t b = align_up(B->arr[a].bytes_per_mask * B->masks_per_batch, 256);
            if (!B->arr[a].want) { B->arr[a].stage[s] = nullptr; continue; }
            if (left < b) return fail(SNAPS_WORKSPACE_TOO_SMALL, "workspace lacks %zu bytes for the staging ring", b - left);
            B->arr[a].stage[s] = r;
            r += b;
            left -= b;
        }
    E->bigk = r;                 // what the ring leaves
    E->bigk_bytes = left;
    const bool knn = B->k > 0;
    const int indeg_arr = 4;
    struct Pending { int m0, nm, buf; };
    Pending prev = {0, 0, -1};
    auto consume = [&](const Pending& pd, int slot) -> snaps_status {
        CUDA_TRY(cudaEventSynchronize(side->copied[slot]));
        snaps_batch_view v;
        memset(&v, 0, sizeof(v));
        v.mask_begin = pd.m0;
        v.mask_end = pd.m0 + pd.nm;
        v.q_begin = j.q_begin;
        v.q_end = j.q_end;
        v.N = j.N;
        v.k = B->k;
        unsigned char* hb = static_cast<unsigned char*>(B->sink->h_buffers[pd.buf]);
        auto at = [&](int a) -> const void* { return B->arr[a].want ? hb + B->arr[a].sink_offset : nullptr; };
        if (knn) {
            v.idx = static_cast<const int32_t*>(at(0));
            v.dist = static_cast<const float*>(at(1));
            v.kth = static_cast<const float*>(at(2));
            v.mean = static_cast<const float*>(at(3));
            v.indeg = static_cast<const int32_t*>(at(4));
        } else {
            v.count = static_cast<const uint32_t*>(at(0));
            v.sumdist = static_cast<const float*>(at(1));
            v.eps_mean = static_cast<const float*>(at(2));
        }
        B->sink->consume(B->sink->user, &v);
        return SNAPS_OK;
    };
    int group = 0;
    for (int m0 = 0; m0 < j.n_masks; m0 += B->masks_per_batch, ++group) {
        const int nm = std::min(B->masks_per_batch, j.n_masks - m0);
        const int s = group & 1;
        // staging slot s is free once its previous copy-out has finished
        if (group >= 2) CUDA_TRY(cudaStreamWaitEvent(E->st, side->copied[s], 0));
        snaps_status rc;
        if (knn) {
            KnnOut o = {reinterpret_cast<int32_t*>(B->arr[0].stage[s]), reinterpret_cast<float*>(B->arr[1].stage[s]),
                        reinterpret_cast<float*>(B->arr[2].stage[s]), reinterpret_cast<float*>(B->arr[3].stage[s]),
                        reinterpret_cast<int32_t*>(B->arr[indeg_arr].stage[s])};
            if (o.indeg) CUDA_TRY(cudaMemsetAsync(o.indeg, 0, B->arr[indeg_arr].bytes_per_mask * nm, E->st));
            if (j.engine == SNAPS_ENGINE_LATTICE)
                rc = lattice_knn_enqueue(E, E->w.batches + (*group_off)[group],
                                         static_cast<int>((*group_off)[group + 1] - (*group_off)[group]), B->k, o);
            else
                rc = grid_knn_enqueue(E, m0, nm, B->k, o);
        } else {
            RangeOut o = {reinterpret_cast<uint32_t*>(B->arr[0].stage[s]), reinterpret_cast<float*>(B->arr[1].stage[s]),
                          reinterpret_cast<float*>(B->arr[2].stage[s])};
            if (j.engine == SNAPS_ENGINE_LATTICE)
                rc = lattice_range_enqueue(E, E->w.batches + (*group_off)[group],
                                           static_cast<int>((*group_off)[group + 1] - (*group_off)[group]), o);
            else
                rc = grid_range_enqueue(E, m0, nm, B->h_eps2, 0, nullptr, o);
        }
        if (rc != SNAPS_OK) return rc;
        CUDA_TRY(cudaEventRecord(side->computed[s], E->st));
        CUDA_TRY(cudaStreamWaitEvent(side->stream, side->computed[s], 0));
        const int buf = B->sink ? group % B->sink->n_buffers : -1;
        for (int a = 0; a < B->n_arr; ++a) {
            if (!B->arr[a].want) continue;
            const size_t bytes = B->arr[a].bytes_per_mask * nm;
            unsigned char* dst = B->sink ? static_cast<unsigned char*>(B->sink->h_buffers[buf]) + B->arr[a].sink_offset
                                         : B->arr[a].h_full + B->arr[a].bytes_per_mask * m0;
            CUDA_TRY(cudaMemcpyAsync(dst, B->arr[a].stage[s], bytes, cudaMemcpyDeviceToHost, side->stream));
        }
        CUDA_TRY(cudaEventRecord(side->copied[s], side->stream));
        if (B->sink) {
            // the previous group is consumed (and its host buffer recycled) while this one computes
            if (group >= 1) {
                rc = consume(prev, (group - 1) & 1);
                if (rc != SNAPS_OK) return rc;
            }
            prev = {m0, nm, buf};
        }
    }
    if (B->sink) {
        snaps_status rc = consume(prev, (group - 1) & 1);
        if (rc != SNAPS_OK) return rc;
    }
    // the caller's stream completes only after the last copies have landed
    for (int s = 0; s < 2 && s < group; ++s) CUDA_TRY(cudaStreamWaitEvent(E->st, side->copied[s], 0));
    return SNAPS_OK;
}

// Plans every mask group of a batched sub-lattice run up front and uploads all descriptors with
// one copy, so that the group loop only enqueues.  Slots are relative to the group's first mask.
snaps_status lattice_plan_groups(Engine* E, const float* thr, int mpb, std::vector<snaps::BatchDesc>* all,
                                 std::vector<size_t>* group_off) {
    const Job& j = E->job;
    for (int m0 = 0; m0 < j.n_masks; m0 += mpb) {
        std::vector<snaps::BatchDesc> b;
        plan_lattice(j.h_masks + m0, std::min(mpb, j.n_masks - m0), thr ? thr + m0 : nullptr, 0, &b);
        group_off->push_back(all->size());
        all->insert(all->end(), b.begin(), b.end());
    }
    group_off->push_back(all->size());
    CUDA_TRY(cudaMemcpyAsync(E->w.batches, all->data(), sizeof(snaps::BatchDesc) * all->size(), cudaMemcpyHostToDevice, E->st));
    return SNAPS_OK;
}

snaps_status sink_check(const snaps_batch_sink* sink, size_t need) {
    if (!sink || !sink->h_buffers || !sink->consume) return fail(SNAPS_INVALID_ARG, "sink, its buffers or its consumer is NULL");
    if (sink->n_buffers < 2) return fail(SNAPS_INVALID_ARG, "sink needs >= 2 host buffers");
    for (int b = 0; b < sink->n_buffers; ++b)
        if (!sink->h_buffers[b]) return fail(SNAPS_INVALID_ARG, "sink buffer %d is NULL", b);
    if (sink->buffer_bytes < need) return fail(SNAPS_INVALID_ARG, "sink buffers hold %zu < %zu bytes", sink->buffer_bytes, need);
    return SNAPS_OK;
}

snaps_status knn_batched(const float* X, int64_t N, int n_feat, int64_t ld, const uint16_t* h_masks, int n_masks, int k,
                         int mpb, int64_t q_begin, int64_t q_end, int flags, void* const h_out[5], const snaps_batch_sink* sink,
                         void* d_ws, size_t ws_bytes, void* stream) {
    prof_reset();
    Engine E;
    E.job = Job{X, N, n_feat, ld, h_masks, n_masks, q_begin, q_end, flags, resolve_engine(flags, N, k)};
    E.st = static_cast<cudaStream_t>(stream);
    snaps_status rc = check_job(E.job, k);
    if (rc) return rc;
    if (k < 1 || k > SNAPS_MAX_K || k > N - 1)
        return fail(SNAPS_INVALID_ARG, "k = %d outside 1..min(N-1, %d)", k, SNAPS_MAX_K);
    if (mpb < 1) return fail(SNAPS_INVALID_ARG, "masks_per_batch < 1");
    const size_t nq = static_cast<size_t>(q_end - q_begin);
    Batched B;
    memset(&B, 0, sizeof(B));
    B.E = &E;
    B.k = k;
    B.masks_per_batch = mpb;
    B.n_arr = 5;
    B.sink = sink;
    const size_t per[5] = {nq * k * 4, nq * k * 4, nq * 4, nq * 4, static_cast<size_t>(N) * 4};
    const unsigned bits[5] = {SNAPS_OUT_IDX, SNAPS_OUT_DIST, SNAPS_OUT_KTH, SNAPS_OUT_MEAN, SNAPS_OUT_INDEG};
    size_t off = 0;
    bool any = false;
    for (int a = 0; a < 5; ++a) {
        B.arr[a].bytes_per_mask = per[a];
        B.arr[a].want = sink ? (sink->want & bits[a]) != 0 : h_out[a] != nullptr;
        B.arr[a].h_full = sink ? nullptr : static_cast<unsigned char*>(h_out[a]);
        B.arr[a].sink_offset = off;
        if (B.arr[a].want) off += align_up(per[a] * mpb, 256);
        any |= B.arr[a].want;
    }
    if (!any) return fail(SNAPS_INVALID_ARG, "no output asked for");
    if (k > snaps::kGridMaxK && (!B.arr[0].want || !B.arr[1].want))
        return fail(SNAPS_INVALID_ARG, "k = %d > %d: the lists are built in place, idx and dist outputs are required", k, snaps::kGridMaxK);
    if (sink) {
        rc = sink_check(sink, off);
        if (rc) return rc;
    }
    rc = carve(d_ws, ws_bytes, E.job, &E.w);
    if (rc) return rc;
    rc = engine_begin(&E);
    if (rc) return rc;
    std::vector<snaps::BatchDesc> all;
    std::vector<size_t> group_off;
    if (E.job.engine == SNAPS_ENGINE_LATTICE) {
        rc = lattice_plan_groups(&E, nullptr, mpb, &all, &group_off);
        if (rc) return rc;
    }
    return run_batched(&B, &all, &group_off);
}

snaps_status range_batched(const float* X, int64_t N, int n_feat, int64_t ld, const uint16_t* h_masks, int n_masks,
                           const float* h_eps, int mpb, int64_t q_begin, int64_t q_end, int flags, const snaps_batch_sink* sink,
                           void* d_ws, size_t ws_bytes, void* stream) {
    prof_reset();
    Engine E;
    E.job = Job{X, N, n_feat, ld, h_masks, n_masks, q_begin, q_end, flags, resolve_engine(flags, N, 0)};
    E.st = static_cast<cudaStream_t>(stream);
    snaps_status rc = check_job(E.job, 0);
    if (rc) return rc;
    if (!h_eps) return fail(SNAPS_INVALID_ARG, "h_eps is NULL");
    if (mpb < 1) return fail(SNAPS_INVALID_ARG, "masks_per_batch < 1");
    std::vector<float> e2, thr;
    rc = eps_squares(h_eps, n_masks, &e2, &thr);
    if (rc) return rc;
    const size_t nq = static_cast<size_t>(q_end - q_begin);
    Batched B;
    memset(&B, 0, sizeof(B));
    B.E = &E;
    B.k = 0;
    B.h_eps2 = e2.data();
    B.masks_per_batch = mpb;
    B.n_arr = 3;
    B.sink = sink;
    const unsigned bits[3] = {SNAPS_OUT_COUNT, SNAPS_OUT_SUMDIST, SNAPS_OUT_EPSMEAN};
    size_t off = 0;
    for (int a = 0; a < 3; ++a) {
        B.arr[a].bytes_per_mask = nq * 4;
        B.arr[a].want = a == 0 || (sink->want & bits[a]) != 0;   // the count drives the kernel: always staged
        B.arr[a].sink_offset = off;
        off += align_up(nq * 4 * mpb, 256);
    }
    rc = sink_check(sink, off);
    if (rc) return rc;
    rc = carve(d_ws, ws_bytes, E.job, &E.w);
    if (rc) return rc;
    rc = engine_begin(&E);
    if (rc) return rc;
    std::vector<snaps::BatchDesc> all;
    std::vector<size_t> group_off;
    if (E.job.engine == SNAPS_ENGINE_LATTICE) {
        rc = lattice_plan_groups(&E, thr.data(), mpb, &all, &group_off);
        if (rc) return rc;
    }
    return run_batched(&B, &all, &group_off);
}

// The radius-grid join of either engine over thresholds already on the device ([n_masks][G]: fl(eps^2) for the
// grid engine, its successor for the sub-lattice engine).
snaps_status range_grid_run(Engine* E, int G, const float* d_thr, const RangeOut& o) {
    const Job& j = E->job;
    if (j.engine == SNAPS_ENGINE_GRID) return grid_range_enqueue(E, 0, j.n_masks, nullptr, G, d_thr, o);
    std::vector<snaps::BatchDesc> batches;
    plan_lattice(j.h_masks, j.n_masks, nullptr, 0, &batches);
    const int nb = static_cast<int>(batches.size());
    CUDA_TRY(cudaMemcpyAsync(E->w.batches, batches.data(), sizeof(snaps::BatchDesc) * nb, cudaMemcpyHostToDevice, E->st));
    CUDA_TRY(cudaMemsetAsync(E->w.counter, 0, 256, E->st));
    snaps::RangeGridParams p;
    p.Xp = E->w.Xp;
    p.Xb = E->w.Xb;
    p.n_blocks = n_blocks_for(j.N);
    p.N = static_cast<int>(j.N);
    p.q_begin = static_cast<int>(j.q_begin);
    p.nq = static_cast<int>(j.nq());
    p.G = G;
    p.batches = E->w.batches;
    p.n_batches = nb;
    p.thr_grid = d_thr;
    p.warps = snaps::kRangeGridMaxThreads / 32;
    while (p.warps > 1 && snaps::range_grid_smem_bytes(G, p.warps) > 227 * 1024) --p.warps;
    p.work_counter = E->w.counter;
    p.out_count = o.count;
    p.out_sum = o.sum;
    p.out_mean = o.mean;
    const int64_t items = static_cast<int64_t>(p.nq) * nb;
    const int grid = static_cast<int>(std::min<int64_t>((items + p.warps - 1) / p.warps, sm_count()));
    const bool prof = prof_begin(E->st);
    CUDA_TRY(snaps::range_grid_launch(p, grid, E->st));
    prof_end(prof, E->st);
    return SNAPS_OK;
}

}  // namespace

// ---- built-in scratch of snaps_knn_selfjoin_static ------------------------------------------
// One array per device that loads the library, held until the process exits.  In host code the
// name below is a host-side stand-in for the symbol, not a device address: the address a kernel
// can use comes from cudaGetSymbolAddress, asked for once per device with that device current.
static __device__ __align__(256) unsigned char g_static_scratch[SNAPS_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
void* g_static_ptr[kMaxDevices] = {};

snaps_status static_scratch_address(void** out) {
    static_assert(SNAPS_STATIC_SCRATCH_BYTES % 256 == 0, "scratch size is a multiple of the carve alignment");
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(SNAPS_UNSUPPORTED, "device ordinal %d outside 0..%d", dev, kMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p) return fail(SNAPS_CUDA_ERROR, "cudaGetSymbolAddress returned a null address");
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return SNAPS_OK;
}

}  // namespace

extern "C" {

const char* snaps_last_error(void) { return g_err; }

const char* snaps_version(void) { return "snaps-b200 0.2 (sm_100a)"; }

size_t snaps_workspace_bytes(int64_t N, int n_feat, int n_masks, int k, int flags) {
    if (N < 2 || N > ((int64_t)1 << 30) || n_feat < 1 || n_feat > SNAPS_MAX_FEATURES || n_masks < 1 || k < 0 || k > SNAPS_MAX_K)
        return 0;
    const int engine = resolve_engine(flags, N, k);
    if (engine != SNAPS_ENGINE_LATTICE && engine != SNAPS_ENGINE_GRID) return 0;
    size_t b = base_workspace_bytes(N, n_feat, n_masks, engine, flags);
    if (engine == SNAPS_ENGINE_GRID && snaps::knn_bigk_pays(N, k) &&
        static_cast<long long>(N) * k <= 0x7fffffffLL)
        b += snaps::knn_bigk_scratch_bytes(N, k);      // long lists on a small table: the selection path's keys
    return b;
}

int64_t snaps_planned_evals(int64_t N, int n_feat, const uint16_t* h_masks, int n_masks) {
    if (!h_masks || n_masks < 1 || N < 2 || n_feat < 1 || n_feat > SNAPS_MAX_FEATURES) return -1;
    std::vector<snaps::BatchDesc> b;
    plan_lattice(h_masks, n_masks, nullptr, 0, &b);
    return static_cast<int64_t>(b.size()) * snaps::kLat * N * N;
}

snaps_status snaps_knn_selfjoin(const float* d_X, int64_t N, int n_feat, int64_t ld,
                                const uint16_t* h_masks, int n_masks, int k, int64_t q_begin, int64_t q_end,
                                int flags, int32_t* out_idx, float* out_dist, float* out_kth, float* out_mean,
                                int32_t* out_indeg, void* d_workspace, size_t workspace_bytes, void* stream) {
    prof_reset();
    Engine E;
    E.job = Job{d_X, N, n_feat, ld, h_masks, n_masks, q_begin, q_end, flags, resolve_engine(flags, N, k)};
    E.st = static_cast<cudaStream_t>(stream);
    snaps_status rc = check_job(E.job, k);
    if (rc) return rc;
    if (k < 1 || k > SNAPS_MAX_K || k > N - 1)
        return fail(SNAPS_INVALID_ARG, "k = %d outside 1..min(N-1, %d)", k, SNAPS_MAX_K);
    if (!out_idx && !out_dist && !out_kth && !out_mean && !out_indeg)
        return fail(SNAPS_INVALID_ARG, "all outputs are NULL");
    if (k > snaps::kGridMaxK && (!out_idx || !out_dist))
        return fail(SNAPS_INVALID_ARG, "k = %d > %d: the lists are built in place, out_idx and out_dist are required", k, snaps::kGridMaxK);
    rc = carve(d_workspace, workspace_bytes, E.job, &E.w);
    if (rc) return rc;
    rc = engine_begin(&E);
    if (rc) return rc;
    if (out_indeg)
        CUDA_TRY(cudaMemsetAsync(out_indeg, 0, sizeof(int32_t) * static_cast<size_t>(n_masks) * N, E.st));
    const KnnOut o = {out_idx, out_dist, out_kth, out_mean, out_indeg};
    E.bigk = E.w.extra;
    E.bigk_bytes = E.w.extra_bytes;
    if (E.job.engine == SNAPS_ENGINE_GRID) return grid_knn_enqueue(&E, 0, n_masks, k, o);
    std::vector<snaps::BatchDesc> batches;
    plan_lattice(h_masks, n_masks, nullptr, 0, &batches);
    CUDA_TRY(cudaMemcpyAsync(E.w.batches, batches.data(), sizeof(snaps::BatchDesc) * batches.size(),
                             cudaMemcpyHostToDevice, E.st));
    return lattice_knn_enqueue(&E, E.w.batches, static_cast<int>(batches.size()), k, o);
}

snaps_status snaps_knn_selfjoin_static(const float* d_X, int64_t N, int n_feat, int64_t ld,
                                       const uint16_t* h_masks, int n_masks, int k, int32_t* out_idx,
                                       float* out_dist, float* out_kth, float* out_mean, int32_t* out_indeg,
                                       void* stream) {
    prof_reset();
    if (N > SNAPS_STATIC_MAX_N)
        return fail(SNAPS_UNSUPPORTED, "N = %lld > %d, the limit of the built-in scratch array (use snaps_knn_selfjoin with a workspace)",
                    (long long)N, SNAPS_STATIC_MAX_N);
    if (n_masks > SNAPS_STATIC_MAX_MASKS)
        return fail(SNAPS_UNSUPPORTED, "n_masks = %d > %d, the limit of the built-in scratch array (use snaps_knn_selfjoin with a workspace)",
                    n_masks, SNAPS_STATIC_MAX_MASKS);
    Engine E;
    E.job = Job{d_X, N, n_feat, ld, h_masks, n_masks, 0, N, SNAPS_ENGINE_LATTICE, SNAPS_ENGINE_LATTICE};
    E.st = static_cast<cudaStream_t>(stream);
    snaps_status rc = check_job(E.job, k);
    if (rc) return rc;
    if (k < 1 || k > SNAPS_LATTICE_MAX_K || k > N - 1)
        return fail(SNAPS_INVALID_ARG, "k = %d outside 1..min(N-1, %d)", k, SNAPS_LATTICE_MAX_K);
    if (!out_idx && !out_dist && !out_kth && !out_mean && !out_indeg)
        return fail(SNAPS_INVALID_ARG, "all outputs are NULL");
    void* scratch = nullptr;
    rc = static_scratch_address(&scratch);
    if (rc) return rc;
    rc = carve(scratch, SNAPS_STATIC_SCRATCH_BYTES, E.job, &E.w);
    if (rc) return rc;
    rc = engine_begin(&E);                  // rewrites every staged row and block the kernel reads
    if (rc) return rc;
    if (out_indeg)
        CUDA_TRY(cudaMemsetAsync(out_indeg, 0, sizeof(int32_t) * static_cast<size_t>(n_masks) * N, E.st));
    const KnnOut o = {out_idx, out_dist, out_kth, out_mean, out_indeg};
    std::vector<snaps::BatchDesc> batches;
    plan_lattice(h_masks, n_masks, nullptr, 0, &batches);
    CUDA_TRY(cudaMemcpyAsync(E.w.batches, batches.data(), sizeof(snaps::BatchDesc) * batches.size(),
                             cudaMemcpyHostToDevice, E.st));
    return lattice_knn_enqueue(&E, E.w.batches, static_cast<int>(batches.size()), k, o);   // zeroes the work counter
}

snaps_status snaps_range_selfjoin(const float* d_X, int64_t N, int n_feat, int64_t ld,
                                  const uint16_t* h_masks, int n_masks, const float* h_eps, int64_t q_begin,
                                  int64_t q_end, int flags, uint32_t* out_count, float* out_sumdist, float* out_mean,
                                  void* d_workspace, size_t workspace_bytes, void* stream) {
    prof_reset();
    Engine E;
    E.job = Job{d_X, N, n_feat, ld, h_masks, n_masks, q_begin, q_end, flags, resolve_engine(flags, N, 0)};
    E.st = static_cast<cudaStream_t>(stream);
    snaps_status rc = check_job(E.job, 0);
    if (rc) return rc;
    if (!h_eps) return fail(SNAPS_INVALID_ARG, "h_eps is NULL");
    if (!out_count) return fail(SNAPS_INVALID_ARG, "out_count is NULL");
    std::vector<float> e2, thr;
    rc = eps_squares(h_eps, n_masks, &e2, &thr);
    if (rc) return rc;
    rc = carve(d_workspace, workspace_bytes, E.job, &E.w);
    if (rc) return rc;
    rc = engine_begin(&E);
    if (rc) return rc;
    const RangeOut o = {out_count, out_sumdist, out_mean};
    if (E.job.engine == SNAPS_ENGINE_GRID) return grid_range_enqueue(&E, 0, n_masks, e2.data(), 0, nullptr, o);
    std::vector<snaps::BatchDesc> batches;
    plan_lattice(h_masks, n_masks, thr.data(), 0, &batches);
    CUDA_TRY(cudaMemcpyAsync(E.w.batches, batches.data(), sizeof(snaps::BatchDesc) * batches.size(),
                             cudaMemcpyHostToDevice, E.st));
    return lattice_range_enqueue(&E, E.w.batches, static_cast<int>(batches.size()), o);
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

snaps_status snaps_range_from_knn(int64_t nq, int n_masks, int k, const float* knn_dist, const float* d_eps,
                                  uint32_t* out_count, float* out_sumdist, float* out_mean, uint8_t* out_complete,
                                  void* stream) {
    if (nq < 1 || n_masks < 1 || k < 1) return fail(SNAPS_INVALID_ARG, "bad sizes");
    if (!knn_dist || !d_eps || !out_count) return fail(SNAPS_INVALID_ARG, "NULL lists, radii or out_count");
    CUDA_TRY(snaps::range_from_knn_launch(nq, n_masks, k, knn_dist, d_eps, out_count, out_sumdist, out_mean, out_complete,
                                          static_cast<cudaStream_t>(stream)));
    return SNAPS_OK;
}

size_t snaps_stream_ring_bytes(int64_t nq, int64_t N, int k, int masks_per_batch) {
    if (nq < 1 || N < 2 || nq > N || k < 0 || masks_per_batch < 1) return 0;
    return ring_bytes(nq, N, k, masks_per_batch);
}

size_t snaps_sink_batch_bytes(int64_t nq, int64_t N, int k, int masks_per_batch, unsigned want) {
    if (nq < 1 || N < 2 || k < 0 || masks_per_batch < 1) return 0;
    const size_t mpb = static_cast<size_t>(masks_per_batch);
    size_t b = 0;
    if (want & SNAPS_OUT_IDX) b += align_up(static_cast<size_t>(nq) * k * 4 * mpb, 256);
    if (want & SNAPS_OUT_DIST) b += align_up(static_cast<size_t>(nq) * k * 4 * mpb, 256);
    if (want & SNAPS_OUT_KTH) b += align_up(static_cast<size_t>(nq) * 4 * mpb, 256);
    if (want & SNAPS_OUT_MEAN) b += align_up(static_cast<size_t>(nq) * 4 * mpb, 256);
    if (want & SNAPS_OUT_INDEG) b += align_up(static_cast<size_t>(N) * 4 * mpb, 256);
    if (want & (SNAPS_OUT_COUNT | SNAPS_OUT_SUMDIST | SNAPS_OUT_EPSMEAN)) b += 3 * align_up(static_cast<size_t>(nq) * 4 * mpb, 256);
    return b;
}

snaps_status snaps_knn_selfjoin_streamed(const float* d_X, int64_t N, int n_feat, int64_t ld,
                                         const uint16_t* h_masks, int n_masks, int k, int masks_per_batch,
                                         int64_t q_begin, int64_t q_end, int flags, int32_t* h_out_idx,
                                         float* h_out_dist, float* h_out_kth, float* h_out_mean,
                                         int32_t* h_out_indeg, void* d_workspace, size_t workspace_bytes, void* stream) {
    void* const h_out[5] = {h_out_idx, h_out_dist, h_out_kth, h_out_mean, h_out_indeg};
    return knn_batched(d_X, N, n_feat, ld, h_masks, n_masks, k, masks_per_batch, q_begin, q_end, flags, h_out, nullptr,
                       d_workspace, workspace_bytes, stream);
}

snaps_status snaps_knn_selfjoin_sink(const float* d_X, int64_t N, int n_feat, int64_t ld, const uint16_t* h_masks,
                                     int n_masks, int k, int masks_per_batch, int64_t q_begin, int64_t q_end, int flags,
                                     const snaps_batch_sink* sink, void* d_workspace, size_t workspace_bytes, void* stream) {
    if (!sink) return fail(SNAPS_INVALID_ARG, "sink is NULL");
    void* const none[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    return knn_batched(d_X, N, n_feat, ld, h_masks, n_masks, k, masks_per_batch, q_begin, q_end, flags, none, sink,
                       d_workspace, workspace_bytes, stream);
}

snaps_status snaps_range_selfjoin_sink(const float* d_X, int64_t N, int n_feat, int64_t ld, const uint16_t* h_masks,
                                       int n_masks, const float* h_eps, int masks_per_batch, int64_t q_begin,
                                       int64_t q_end, int flags, const snaps_batch_sink* sink, void* d_workspace,
                                       size_t workspace_bytes, void* stream) {
    if (!sink) return fail(SNAPS_INVALID_ARG, "sink is NULL");
    return range_batched(d_X, N, n_feat, ld, h_masks, n_masks, h_eps, masks_per_batch, q_begin, q_end, flags, sink,
                         d_workspace, workspace_bytes, stream);
}

size_t snaps_range_grid_workspace_bytes(int64_t N, int n_feat, int n_masks, int G, int flags) {
    if (N < 2 || n_feat < 1 || n_feat > SNAPS_MAX_FEATURES || n_masks < 1 || G < 1 || G > snaps::kRangeGridMaxRadii)
        return 0;
    const int engine = resolve_engine(flags, N, 0);
    if (engine != SNAPS_ENGINE_LATTICE && engine != SNAPS_ENGINE_GRID) return 0;
    return base_workspace_bytes(N, n_feat, n_masks, engine, flags) + align_up(static_cast<size_t>(n_masks) * G * 4, 256);
}

snaps_status snaps_range_selfjoin_grid(const float* d_X, int64_t N, int n_feat, int64_t ld,
                                       const uint16_t* h_masks, int n_masks, const float* h_eps_grid, int G,
                                       int64_t q_begin, int64_t q_end, int flags, uint32_t* out_count,
                                       float* out_sumdist, float* out_mean, void* d_workspace, size_t workspace_bytes,
                                       void* stream) {
    prof_reset();
    Engine E;
    E.job = Job{d_X, N, n_feat, ld, h_masks, n_masks, q_begin, q_end, flags, resolve_engine(flags, N, 0)};
    E.st = static_cast<cudaStream_t>(stream);
    snaps_status rc = check_job(E.job, 0);
    if (rc) return rc;
    if (!h_eps_grid || !out_count) return fail(SNAPS_INVALID_ARG, "NULL eps grid or out_count");
    if (G < 1 || G > snaps::kRangeGridMaxRadii) return fail(SNAPS_INVALID_ARG, "G = %d outside 1..%d", G, snaps::kRangeGridMaxRadii);
    const bool grid_engine = E.job.engine == SNAPS_ENGINE_GRID;
    std::vector<float> thr(static_cast<size_t>(n_masks) * G);
    for (int m = 0; m < n_masks; ++m)
        for (int g = 0; g < G; ++g) {
            const float e = h_eps_grid[static_cast<size_t>(m) * G + g];
            if (!(e > 0.f) || !isfinite(e) || (g > 0 && !(e > h_eps_grid[static_cast<size_t>(m) * G + g - 1])))
                return fail(SNAPS_INVALID_ARG, "eps_grid[%d][%d] = %g: radii must be finite, > 0 and ascending", m, g, (double)e);
            const float e2 = static_cast<float>(static_cast<double>(e) * static_cast<double>(e));
            // closed ball, reading A2: d^2 <= fl(eps^2) (grid engine) <=> d^2 < nextafter (sub-lattice engine)
            thr[static_cast<size_t>(m) * G + g] = grid_engine ? e2 : nextafterf(e2, INFINITY);
        }
    rc = carve(d_workspace, workspace_bytes, E.job, &E.w);
    if (rc) return rc;
    rc = engine_begin(&E);
    if (rc) return rc;
    const size_t grid_bytes = align_up(static_cast<size_t>(n_masks) * G * 4, 256);
    if (E.w.extra_bytes < grid_bytes)
        return fail(SNAPS_WORKSPACE_TOO_SMALL, "workspace lacks %zu bytes for the radius grid", grid_bytes);
    // pageable host source: the copy is staged before cudaMemcpyAsync returns
    CUDA_TRY(cudaMemcpyAsync(E.w.extra, thr.data(), thr.size() * 4, cudaMemcpyHostToDevice, E.st));
    return range_grid_run(&E, G, reinterpret_cast<const float*>(E.w.extra), RangeOut{out_count, out_sumdist, out_mean});
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
    const Job job = Job{d_X, N, n_feat, ld, h_masks, n_masks, 0, N, 0, SNAPS_ENGINE_LATTICE};
    snaps_status rc = check_job(job, 0);
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

size_t snaps_eps_search_workspace_bytes(int nq, int nc, int n_masks, int n_bins, int n_targets) {
    if (nq < 1 || nc < 1 || n_masks < 1 || n_bins < 1 || n_bins > 8192 || n_targets < 1) return 0;
    return snaps::eps_search_workspace_bytes(nq, nc, n_masks, n_bins, n_targets);
}

snaps_status snaps_eps_search(const float* d_X, int64_t N, int n_feat, int64_t ld, const uint16_t* h_masks, int n_masks,
                              const int32_t* h_sample_q, int nq, const int32_t* h_sample_c, int nc, int n_bins,
                              const double* h_target_s, int n_targets, float* out_eps_mean, float* out_eps,
                              unsigned long long* out_hist, void* d_workspace, size_t workspace_bytes, void* stream) {
    const Job job = Job{d_X, N, n_feat, ld, h_masks, n_masks, 0, N, 0, SNAPS_ENGINE_LATTICE};
    snaps_status rc = check_job(job, 0);
    if (rc) return rc;
    if (!h_sample_q || !h_sample_c || !h_target_s || !out_eps_mean || !out_eps || nq < 1 || nc < 1 || n_targets < 1)
        return fail(SNAPS_INVALID_ARG, "NULL or empty samples, targets or outputs");
    if (n_bins < 1 || n_bins > 8192) return fail(SNAPS_INVALID_ARG, "n_bins = %d outside 1..8192", n_bins);
    for (int t = 0; t < n_targets; ++t)
        if (!(h_target_s[t] > 0.0)) return fail(SNAPS_INVALID_ARG, "target selectivity %d is not > 0", t);
    // pairs with c != q: both samples are id lists; count the ids they share
    std::vector<int32_t> a(h_sample_q, h_sample_q + nq), b(h_sample_c, h_sample_c + nc);
    for (int32_t v : a) if (v < 0 || v >= N) return fail(SNAPS_INVALID_ARG, "query sample id out of range");
    for (int32_t v : b) if (v < 0 || v >= N) return fail(SNAPS_INVALID_ARG, "candidate sample id out of range");
    std::sort(a.begin(), a.end());
    std::sort(b.begin(), b.end());
    if (std::adjacent_find(a.begin(), a.end()) != a.end() || std::adjacent_find(b.begin(), b.end()) != b.end())
        return fail(SNAPS_INVALID_ARG, "sample ids must be distinct");
    std::vector<int32_t> both;
    std::set_intersection(a.begin(), a.end(), b.begin(), b.end(), std::back_inserter(both));
    const long long pairs = static_cast<long long>(nq) * nc - static_cast<long long>(both.size());
    if (pairs < 1) return fail(SNAPS_INVALID_ARG, "no sampled pair with c != q");
    if (!d_workspace || workspace_bytes < snaps::eps_search_workspace_bytes(nq, nc, n_masks, n_bins, n_targets))
        return fail(SNAPS_WORKSPACE_TOO_SMALL, "eps search workspace too small");
    CUDA_TRY(snaps::eps_search_launch(d_X, N, ld, n_feat, h_sample_q, nq, h_sample_c, nc, pairs, h_masks, n_masks, n_bins,
                                      h_target_s, n_targets, out_eps_mean, out_eps, out_hist, d_workspace,
                                      static_cast<cudaStream_t>(stream)));
    return SNAPS_OK;
}

// ---- DSSJ parameter selection in one call --------------------------------
namespace {
struct SelectEpsLayout {
    size_t search, mm, grid, thr, score, order, u, rank, total;
};
SelectEpsLayout select_eps_layout(int64_t N, int n_masks, int G, int nq, int nc, int n_bins) {
    SelectEpsLayout L;
    const size_t rows = static_cast<size_t>(n_masks) * G;
    L.search = align_up(snaps::eps_search_workspace_bytes(nq, nc, n_masks, n_bins, 2), 256);
    L.mm = align_up(static_cast<size_t>(n_masks) * 3 * 4, 256);          // eps_mean, then (eps_min, eps_max) pairs
    L.grid = align_up(rows * 4, 256);
    L.thr = align_up(rows * 4, 256);
    L.score = align_up(rows * static_cast<size_t>(N) * 4, 256);          // x3: count, sum, mean
    L.order = align_up(rows * static_cast<size_t>(N) * 4, 256);
    L.u = align_up(sizeof(float) * 4 * rows, 256);
    L.rank = align_up(snaps::rank_workspace_bytes(N, static_cast<int>(rows)), 256);
    L.total = L.search + L.mm + L.grid + L.thr + 3 * L.score + L.order + L.u + L.rank;
    return L;
}
}  // namespace

size_t snaps_select_eps_workspace_bytes(int64_t N, int n_feat, int n_masks, int G, int nq, int nc, int n_bins, int flags) {
    if (N < 2 || n_feat < 1 || n_feat > SNAPS_MAX_FEATURES || n_masks < 1 || G < 2 || G > snaps::kRangeGridMaxRadii ||
        nq < 1 || nc < 1 || n_bins < 1 || n_bins > 8192)
        return 0;
    const int engine = resolve_engine(flags, N, 0);
    if (engine != SNAPS_ENGINE_LATTICE && engine != SNAPS_ENGINE_GRID) return 0;
    return base_workspace_bytes(N, n_feat, n_masks, engine, flags) + select_eps_layout(N, n_masks, G, nq, nc, n_bins).total;
}

snaps_status snaps_range_select_eps(const float* d_X, int64_t N, int n_feat, int64_t ld, const uint16_t* h_masks,
                                    int n_masks, const int32_t* h_sample_q, int nq, const int32_t* h_sample_c, int nc,
                                    int n_bins, double s_min, double s_max, int G, int n_top, int flags,
                                    float* out_eps_grid, int32_t* out_j_count, int32_t* out_j_mean, float* out_u,
                                    void* d_workspace, size_t workspace_bytes, void* stream) {
    prof_reset();
    Engine E;
    E.job = Job{d_X, N, n_feat, ld, h_masks, n_masks, 0, N, flags, resolve_engine(flags, N, 0)};
    E.st = static_cast<cudaStream_t>(stream);
    snaps_status rc = check_job(E.job, 0);
    if (rc) return rc;
    if (flags & SNAPS_FLAG_X_ON_HOST) return fail(SNAPS_UNSUPPORTED, "snaps_range_select_eps takes a device table");
    if (G < 2 || G > snaps::kRangeGridMaxRadii) return fail(SNAPS_INVALID_ARG, "G = %d outside 2..%d", G, snaps::kRangeGridMaxRadii);
    if (!(s_min > 0.0) || !(s_max > s_min)) return fail(SNAPS_INVALID_ARG, "need 0 < s_min < s_max");
    if (n_top < 1 || n_top > N) return fail(SNAPS_INVALID_ARG, "n_top = %d outside 1..N", n_top);
    if (!out_j_count || !out_j_mean) return fail(SNAPS_INVALID_ARG, "NULL outputs");
    if ((N + 31) / 32 * 4 > 200 * 1024) return fail(SNAPS_UNSUPPORTED, "N too large for the top-n bitmap");
    rc = carve(d_workspace, workspace_bytes, E.job, &E.w);
    if (rc) return rc;
    const SelectEpsLayout L = select_eps_layout(N, n_masks, G, nq, nc, n_bins);
    if (E.w.extra_bytes < L.total) return fail(SNAPS_WORKSPACE_TOO_SMALL, "workspace lacks %zu bytes", L.total - E.w.extra_bytes);
    unsigned char* p = E.w.extra;
    void* search_ws = p; p += L.search;
    float* eps_mean = reinterpret_cast<float*>(p);
    float* eps_mm = eps_mean + n_masks; p += L.mm;
    float* eps_grid = reinterpret_cast<float*>(p); p += L.grid;
    float* thr = reinterpret_cast<float*>(p); p += L.thr;
    uint32_t* count = reinterpret_cast<uint32_t*>(p); p += L.score;
    float* sum = reinterpret_cast<float*>(p); p += L.score;
    float* mean = reinterpret_cast<float*>(p); p += L.score;
    int32_t* order = reinterpret_cast<int32_t*>(p); p += L.order;
    float* u = out_u ? out_u : reinterpret_cast<float*>(p); p += L.u;
    void* rws = p;
    // 1. eps_min, eps_max for the two target selectivities (NEXT-2)
    const double targets[2] = {s_min, s_max};
    rc = snaps_eps_search(d_X, N, n_feat, ld, h_masks, n_masks, h_sample_q, nq, h_sample_c, nc, n_bins, targets, 2, eps_mean,
                          eps_mm, nullptr, search_ws, L.search, stream);
    if (rc) return rc;
    // 2. the eps grid and its squared thresholds
    CUDA_TRY(snaps::eps_grid_launch(eps_mm, n_masks, G, E.job.engine == SNAPS_ENGINE_LATTICE ? 1 : 0, eps_grid, thr, E.st));
    if (out_eps_grid)
        CUDA_TRY(cudaMemcpyAsync(out_eps_grid, eps_grid, sizeof(float) * static_cast<size_t>(n_masks) * G, cudaMemcpyDeviceToDevice, E.st));
    // 3. one join at eps_max gives every eps_j
    rc = engine_begin(&E);
    if (rc) return rc;
    rc = range_grid_run(&E, G, thr, RangeOut{count, sum, mean});
    if (rc) return rc;
    // 4. ranks, Eq. 2 against the smallest and the largest radius, Eq. 3 -- for both DSSJ metrics
    const int rows = n_masks * G;
    for (int metric = 0; metric < 2; ++metric) {
        const int kind = metric == 0 ? SNAPS_METRIC_DSSJ_COUNT : SNAPS_METRIC_DSSJ_MEAN;
        float* u_min = u + static_cast<size_t>(2 * metric) * rows;
        float* u_max = u + static_cast<size_t>(2 * metric + 1) * rows;
        CUDA_TRY(snaps::rank_launch(kind, metric == 0 ? static_cast<const void*>(count) : static_cast<const void*>(mean), count, N,
                                    rows, nullptr, order, rws, L.rank, E.st));
        for (int g = 0; g < G; ++g) {
            CUDA_TRY(snaps::topn_overlap_strided_launch(order, order, N, n_masks, n_top, G, 0, G, g,
                                                        u_min + static_cast<size_t>(g) * n_masks, E.st));
            CUDA_TRY(snaps::topn_overlap_strided_launch(order, order, N, n_masks, n_top, G, G - 1, G, g,
                                                        u_max + static_cast<size_t>(g) * n_masks, E.st));
        }
        CUDA_TRY(snaps::select_launch(u_min, u_max, G, n_masks, n_top, metric == 0 ? out_j_count : out_j_mean, E.st));
    }
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

size_t snaps_select_k_workspace_bytes(int64_t N, int n_masks, int G) {
    if (N < 2 || n_masks < 1 || G < 2 || G > 256) return 0;
    const size_t arr = align_up(static_cast<size_t>(N) * n_masks * 4, 256);
    // score array, three order arrays (smallest k, largest k, current k), the U curves, ranking scratch
    return 4 * arr + align_up(sizeof(float) * 4 * G * static_cast<size_t>(n_masks), 256) +
           align_up(snaps::rank_workspace_bytes(N, n_masks), 256);
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
    if (!d_workspace || workspace_bytes < snaps_select_k_workspace_bytes(N, n_masks, G))
        return fail(SNAPS_WORKSPACE_TOO_SMALL, "workspace %zu < %zu bytes", workspace_bytes,
                    snaps_select_k_workspace_bytes(N, n_masks, G));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t arr = align_up(static_cast<size_t>(N) * n_masks * 4, 256);
    unsigned char* p = static_cast<unsigned char*>(d_workspace);
    void* score = p;
    int32_t* ord_min = reinterpret_cast<int32_t*>(p + arr);
    int32_t* ord_max = reinterpret_cast<int32_t*>(p + 2 * arr);
    int32_t* ord_cur = reinterpret_cast<int32_t*>(p + 3 * arr);
    const size_t u_bytes = align_up(sizeof(float) * 4 * G * static_cast<size_t>(n_masks), 256);
    void* rws = p + 4 * arr + u_bytes;
    const size_t rws_bytes = workspace_bytes - 4 * arr - u_bytes;
    float* u = out_u ? out_u : reinterpret_cast<float*>(p + 4 * arr);   // U curves: the caller's array or the workspace
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
    g_prof.on = on != 0;
    prof_reset();
    return SNAPS_OK;
}

snaps_status snaps_profile_last_kernel_ms(float* h_ms, int* h_launches) {
    float total = 0.f;
    for (size_t i = 0; i < g_prof.used; ++i) {
        CUDA_TRY(cudaEventSynchronize(g_prof.pool[i].second));
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, g_prof.pool[i].first, g_prof.pool[i].second));
        total += ms;
    }
    if (h_ms) *h_ms = total;
    if (h_launches) *h_launches = static_cast<int>(g_prof.used);
    return SNAPS_OK;
}

snaps_status snaps_probe_fp32_rate(int kind, double* h_lane_ops_per_s, void* d_scratch, void* stream) {
    if (kind < 0 || kind > 5 || !h_lane_ops_per_s || !d_scratch) return fail(SNAPS_INVALID_ARG, "bad probe arguments");
    double ops = 0.0;
    float ms = 0.f;
    CUDA_TRY(snaps::probe_fp32_launch(kind, &ops, &ms, static_cast<float*>(d_scratch), static_cast<cudaStream_t>(stream)));
    *h_lane_ops_per_s = ops / (static_cast<double>(ms) * 1e-3);
    return SNAPS_OK;
}

}  // extern "C"
