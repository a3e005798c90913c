// knn_lattice.cu -- kNN self-join over a batch of feature subspaces (steps a3-a5, a7).
//
// What it computes: PAPER.md:112, 122 (kNNSJ) for every mask of a sub-lattice batch;
// scores of PAPER.md:251-252 fused into the tail.  How:
//   * one warp = one query object x the 64 masks {H u T : T subset of features 0..5};
//     the 32 lanes hold 32 different candidates per step;
//   * candidates stream from the blocked copy of the table (2 MB at N=31,693: L2 resident,
//     four coalesced 128-bit loads per step, next block prefetched into registers); no barrier
//     couples the warps of a CTA;
//   * FILTER (every candidate, snaps_device.cuh: lattice_filter): squared differences once, then the
//     16 partial sums X[u] over features 2..5 (add-only).  X[u] is a lower bound of the four sums
//     X[u] (+sq0) (+sq1) of "group" u (adding non-negative terms never rounds below the
//     addend), so a candidate can enter one of the group's lists only if X[u] < G[u],
//     G[u] = max of the group's four current thresholds (register-held);
//   * COMPACT: lanes that pass any group test push (id, base, sq0..5) into a per-warp
//     shared-memory queue (ballot + popc); with running thresholds a few % of candidates pass;
//   * EXACT TEST (every 32 queued candidates, lane = candidate): the 64 subset sums by add-only
//     enumeration in a fixed order, each compared with its list's current threshold (broadcast reads);
//     about one queued candidate in four has a sum that can enter a list -- only those wait for
//   * REFINE (every 32 survivors, all lanes busy): lane = candidate forms the 64 sums again; they
//     cross to the list owners through a 32 x 32 shared-memory transpose; lane = list merges the
//     sums below its threshold into its sorted list, held in registers for the merge (right-aligned,
//     branch-free insert); a list is 12/20/28/36 words apart from the next so that whole lists move
//     with conflict-free 128-bit accesses; thresholds and G are refreshed;
//   * thresholds start from an upper bound seeded by evaluating k known objects
//     (the first k ids or the previous batch's neighbours: consecutive batches
//     differ in one feature), tightened by min over supersets (the k-th distance
//     is monotone in the feature set).
#include "knn_lattice.cuh"

namespace snaps {


// ---- per-warp shared-memory state (32-bit words); S = list stride (template parameter) ----
//   [0, 64*S)        list d^2, list L at L*S, ascending by (d^2, id), right aligned
//   [64*S, 128*S)    list ids
//   then rows of 64 words: (unused), threshold, seed bound, output slot,
//   one row: words 0..15 G (group maxima), words 16..30 the query's 15 features
//   then the 32 x 32 transpose (row stride 36), the candidate ids of a refine step and the
//   queue (kQueue entries of 8 words)
#define L_D2(e, L) ws[(L) * S + (e)]
#define L_ID(e, L) wsi[64 * S + (L) * S + (e)]
#define ROWS(r) (128 * S + (r) * 64)
#define THR(L) ws[ROWS(1) + (L)]
#define SEED(L) ws[ROWS(2) + (L)]
#define SLOT(L) wsi[ROWS(3) + (L)]
#define GMAX(u) ws[ROWS(4) + (u)]
#define QROW(j) ws[ROWS(4) + 16 + (j)]
#define MT(T, j) ws[ROWS(5) + (T) * 36 + (j)]
#define CANDID(j) wsi[ROWS(5) + 32 * 36 + (j)]
#define QUEUE4 (reinterpret_cast<float4*>(ws + ROWS(5) + 32 * 36 + 32))
constexpr int kQueue = 64;   // queue entries (8 words each); exact test as soon as 32 are waiting
// the candidates that passed the exact test wait here for the refine step, at most 32 of them: the
// refine step takes them all into registers before it writes the transpose, so the two share storage
#define SURV4 (reinterpret_cast<float4*>(&MT(0, 0)))

__host__ __device__ constexpr int knn_list_stride(int k) { return k <= 12 ? 12 : k <= 20 ? 20 : k <= 28 ? 28 : 36; }
__host__ __device__ constexpr int knn_warp_words(int k) {
    return 128 * knn_list_stride(k) + 5 * 64 + 32 * 36 + 32 + kQueue * 8;
}

// REFINE: lanes 0..n-1 take the n waiting survivors of the exact test and form their 64 subset sums
// (lane = candidate); the sums cross to the list owners through a 32 x 32 shared-memory
// transpose (row stride 36 words: conflict-free both ways), 32 lists at a time; then
// lane = list: the owner compares its list's 32 new sums with its threshold and merges the
// passing ones into the sorted list held in registers (rank computation, no shift loop).
// Candidates come in increasing id order, so among equal d^2 the earlier one stays first:
// ties are broken by the smaller id (reading A3).
// The add order (high features by FMA in feature order -> features 2,3,4,5 -> 0 -> 1) is the
// same wherever a squared distance is formed, so a value never depends on scheduling.
template <int S>
__device__ __noinline__ void knn_refine(float* ws, int k, int lane, int n) {
    constexpr int NE = S > 32 ? 32 : S;   // list elements held (S = 36 carries 4 words of padding)
    int* wsi = reinterpret_cast<int*>(ws);
    __syncwarp();
    PairTerms pt;
    const int cand = survivors_pop(SURV4, lane, n, pt);
    __syncwarp();   // the transpose overwrites the survivors' storage
    CANDID(lane) = cand;
    float X8[8];   // partial sums over features 2,3,4; feature 5 is added per half (same order as X[16])
    lattice_partial8(pt, X8);
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        lattice_sums_to_transpose(pt, X8, half, &MT(0, 0), lane);
        __syncwarp();
        // ---- lane = list T.  The k entries are right aligned in the NE slots (ascending; unused
        // bottom slots hold -inf, not yet filled top slots +inf), so the k-th is always slot NE-1.
        const int T = 32 * half + lane;
        const float seed = SEED(T);
        float thr = THR(T);
        bool changed = false;
        float v[NE];
        int w[NE];
        {
            const float4* pv = reinterpret_cast<const float4*>(&L_D2(0, T));
            const int4* pw = reinterpret_cast<const int4*>(&L_ID(0, T));
#pragma unroll
            for (int e4 = 0; e4 < NE / 4; ++e4) {
                const float4 a = pv[e4];
                const int4 b = pw[e4];
                v[4 * e4 + 0] = a.x; v[4 * e4 + 1] = a.y; v[4 * e4 + 2] = a.z; v[4 * e4 + 3] = a.w;
                w[4 * e4 + 0] = b.x; w[4 * e4 + 1] = b.y; w[4 * e4 + 2] = b.z; w[4 * e4 + 3] = b.w;
            }
        }
        // which of the 32 new sums can enter (against the threshold as it stands now) ...
        unsigned mask = 0u;
#pragma unroll
        for (int j4 = 0; j4 < 8; ++j4) {
            const float4 m = *reinterpret_cast<const float4*>(&MT(lane, 4 * j4));
            mask |= (m.x < thr ? 1u : 0u) << (4 * j4);
            mask |= (m.y < thr ? 1u : 0u) << (4 * j4 + 1);
            mask |= (m.z < thr ? 1u : 0u) << (4 * j4 + 2);
            mask |= (m.w < thr ? 1u : 0u) << (4 * j4 + 3);
        }
        // ... merged in candidate order (= increasing id).  Every id already in the list is
        // smaller than the new one, so "list entry e precedes (d, id)" is v[e] <= d, and the
        // new sorted array is v'[e] = v[e] if v[e] <= d, else d if v[e-1] <= d, else v[e-1].
#pragma unroll 1
        while (mask) {
            const int j = __ffs(mask) - 1;
            mask &= mask - 1u;
            const float d = MT(lane, j);
            const int id = CANDID(j);
            if (d < thr) {
                changed = true;
                bool below[NE];
#pragma unroll
                for (int e = 0; e < NE; ++e) below[e] = v[e] <= d;
#pragma unroll
                for (int e = NE - 1; e >= 1; --e) {
                    v[e] = below[e] ? v[e] : (below[e - 1] ? d : v[e - 1]);
                    w[e] = below[e] ? w[e] : (below[e - 1] ? id : w[e - 1]);
                }
                v[0] = below[0] ? v[0] : d;
                w[0] = below[0] ? w[0] : id;
                thr = fminf(seed, v[NE - 1]);
            }
        }
        if (changed) {
            float4* qv = reinterpret_cast<float4*>(&L_D2(0, T));
            int4* qw = reinterpret_cast<int4*>(&L_ID(0, T));
#pragma unroll
            for (int e4 = 0; e4 < NE / 4; ++e4) {
                qv[e4] = make_float4(v[4 * e4], v[4 * e4 + 1], v[4 * e4 + 2], v[4 * e4 + 3]);
                qw[e4] = make_int4(w[4 * e4], w[4 * e4 + 1], w[4 * e4 + 2], w[4 * e4 + 3]);
            }
            THR(T) = thr;
        }
        __syncwarp();
    }
    if (lane < 16) {
        const float4 t = *reinterpret_cast<const float4*>(&THR(4 * lane));
        GMAX(lane) = fmaxf(fmaxf(t.x, t.y), fmaxf(t.z, t.w));
    }
    __syncwarp();
}

// EXACT TEST of 32 queued candidates against the 64 current thresholds (snaps_device.cuh).
template <int S>
__device__ __noinline__ int knn_exact_test(float* ws, int lane, int q, int N, int head, int n, int nb) {
    __syncwarp();
    return lattice_exact_test(QUEUE4, kQueue, SURV4, &THR(0), lane, q, N, head, n, nb);
}

// Upper bounds on the final k-th squared distance of every list of the new batch.
template <int S>
__device__ __noinline__ void knn_seed(float* ws, const float* __restrict__ Xp, int q, int k,
                                      uint32_t H, bool has_prev, int lane) {
    constexpr int NE = S > 32 ? 32 : S;
    int* wsi = reinterpret_cast<int*>(ws);
    __syncwarp();
    float qrow[15];
#pragma unroll
    for (int j = 0; j < 15; ++j) qrow[j] = QROW(j);
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
        const int L = lane + 32 * h;
        float bound = -1.f;
        if (SLOT(L) >= 0) {
            const uint32_t mask = H | static_cast<uint32_t>(L);
            // k known objects bound the k-th distance: the previous batch's neighbours of this slot
            // (consecutive batches differ in one feature) if that list is full, else the first k ids
            const bool from_prev = has_prev && L_D2(NE - 1, L) < __int_as_float(0x7f800000);
            float b1 = 0.f;
            // two rows in flight per lane: the loads are scattered (L2 latency) and nothing else hides them
#pragma unroll 1
            for (int e = 0; e < k; e += 2) {
                const int e1 = min(e + 1, k - 1);
                const int c0 = from_prev ? L_ID(NE - k + e, L) : e + (e >= q ? 1 : 0);
                const int c1 = from_prev ? L_ID(NE - k + e1, L) : e1 + (e1 >= q ? 1 : 0);
                const float d0 = masked_d2(Xp + static_cast<size_t>(c0) * kRowFloats, qrow, mask);
                const float d1 = masked_d2(Xp + static_cast<size_t>(c1) * kRowFloats, qrow, mask);
                b1 = fmaxf(b1, fmaxf(d0, d1));
            }
            bound = b1;
            // the stream re-evaluates these objects in another summation order: leave
            // room for rounding (<= 15 * 2^-24 relative) so that none of them is lost
            bound = fmaxf(bound * 1.00002f, 1e-30f);
        }
        SEED(L) = bound;
    }
    __syncwarp();
    // D_(k)(S) <= D_(k)(S u {f}): a superset's bound also bounds the subset
#pragma unroll 1
    for (int bit = 0; bit < kLow; ++bit) {
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            const int L = lane + 32 * h;
            if (!((L >> bit) & 1)) {
                const float a = SEED(L), b = SEED(L | (1 << bit));
                if (a >= 0.f && b >= 0.f) SEED(L) = fminf(a, b);
            }
        }
        __syncwarp();
    }
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
        const int L = lane + 32 * h;
        // empty list: k right-aligned slots at +inf above NE-k slots at -inf
        for (int e = 0; e < NE; ++e)
            L_D2(e, L) = __int_as_float(e < NE - k ? 0xff800000 : 0x7f800000);
        THR(L) = SEED(L);
    }
    __syncwarp();
    if (lane < 16) {
        const float4 t = *reinterpret_cast<const float4*>(&THR(4 * lane));
        GMAX(lane) = fmaxf(fmaxf(t.x, t.y), fmaxf(t.z, t.w));
    }
    __syncwarp();
}

// Step a7: sqrt, scores, in-degree, lists.
template <int S>
__device__ __noinline__ void knn_emit(float* ws, const KnnParams& p, int q, int lane) {
    constexpr int NE = S > 32 ? 32 : S;
    int* wsi = reinterpret_cast<int*>(ws);
    const int k = p.k;
    __syncwarp();
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
        const int L = lane + 32 * h;
        const int sl = SLOT(L);
        if (sl < 0) continue;
        const size_t o = static_cast<size_t>(sl) * static_cast<size_t>(p.nq) + static_cast<size_t>(q - p.q_begin);
        float sum = 0.f, dk = 0.f;
#pragma unroll 1
        for (int e = 0; e < k; ++e) {
            const float d = sqrtf(L_D2(NE - k + e, L));
            const int id = L_ID(NE - k + e, L);
            sum += d;
            dk = d;
            // streaming stores: the outputs are written once and must not push the in-degree rows of the
            // batches in flight (L2-resident atomics) out of the L2
            if (p.out_idx) __stcs(&p.out_idx[o * k + e], id);
            if (p.out_dist) __stcs(&p.out_dist[o * k + e], d);
            if (p.out_indeg)
                atomicAdd(&p.out_indeg[static_cast<size_t>(sl) * static_cast<size_t>(p.N) + id], 1);
        }
        if (p.out_kth) __stcs(&p.out_kth[o], dk);
        if (p.out_mean) __stcs(&p.out_mean[o], sum / static_cast<float>(k));
    }
    __syncwarp();
}

#define RELOAD_G()                                                            \
    do {                                                                      \
        const float4* g4_ = reinterpret_cast<const float4*>(&GMAX(0));        \
        _Pragma("unroll") for (int i4 = 0; i4 < 4; ++i4) {                    \
            const float4 v = g4_[i4];                                         \
            G[4 * i4 + 0] = v.x;                                              \
            G[4 * i4 + 1] = v.y;                                              \
            G[4 * i4 + 2] = v.z;                                              \
            G[4 * i4 + 3] = v.w;                                              \
        }                                                                     \
    } while (0)

// Every candidate block in id order (the table is L2 resident at the sizes this engine serves;
// large tables and arbitrary mask lists take the grid engine, grid_join.cu).
template <int S>
__global__ void __launch_bounds__(kKnnMaxThreads, 1) knn_lattice_kernel(const KnnParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int k = p.k;
    float* ws = reinterpret_cast<float*>(smem + 128) + static_cast<size_t>(warp) * knn_warp_words(k);
    int* wsi = reinterpret_cast<int*>(ws);

    // one item = one query x a run of consecutive batches, fetched per warp: no block-level
    // synchronisation anywhere in the kernel (a warp never waits for a slower query)
    const long long n_items = static_cast<long long>(p.nq) * p.n_bchunks;
    const unsigned lt = (1u << lane) - 1u;
    const int n_blocks = p.n_blocks;
    for (;;) {
        long long item = 0;
        if (lane == 0) item = atomicAdd(p.work_counter, 1ull);
        item = __shfl_sync(kFull, item, 0);
        if (item >= n_items) break;
        const int q = p.q_begin + static_cast<int>(item % p.nq);
        const int bc = static_cast<int>(item / p.nq);
        const int b0 = bc * p.batches_per_item;
        const int b1 = min(b0 + p.batches_per_item, p.n_batches);

        FilterQuery fq;
        float qhi[9];
        {
            const float* qr = p.Xp + static_cast<size_t>(q) * kRowFloats;
            float qlo[kLow];
#pragma unroll
            for (int j = 0; j < kLow; ++j) qlo[j] = qr[j];
            filter_query_set_row(fq, qlo);
#pragma unroll
            for (int j = 0; j < 9; ++j) qhi[j] = qr[kLow + j];
            if (lane < 15) QROW(lane) = qr[lane];
        }
        bool has_prev = false;
#pragma unroll 1
        for (int b = b0; b < b1; ++b) {
            const BatchDesc* bd = &p.batches[b];
            const uint32_t H = bd->hmask;
            SLOT(lane) = bd->slot[lane];
            SLOT(lane + 32) = bd->slot[lane + 32];
            knn_seed<S>(ws, p.Xp, q, k, H, has_prev, lane);
            filter_query_init(fq, qhi, H);
            float G[16];
            RELOAD_G();
            int qhead = 0, qtail = 0;  // queue positions (warp-uniform, monotone)
            int nsurv = 0;             // candidates waiting for the refine step
            // candidates: block t = rows 32t..32t+31, lane = row, four coalesced 128-bit loads;
            // two register sets alternate (one in use, one in flight) -- no register moves
#define FILTER_BLOCK(r, t_)                                                                   \
    {                                                                                         \
        PairTerms pt;                                                                         \
        const bool pass = lattice_filter<G0>(r, fq, G, pt);                                   \
        const unsigned bal = __ballot_sync(kFull, pass);                                      \
        if (bal) {                                                                            \
            qtail += queue_push(QUEUE4, kQueue, qtail, pass, bal, lt, (t_) * 32 + lane, pt);  \
            while (qtail - qhead >= 32) {                                                     \
                const int r_ = knn_exact_test<S>(ws, lane, q, p.N, qhead, 32, nsurv);         \
                qhead += r_ & 0xff;                                                           \
                nsurv = r_ >> 8;                                                              \
                if (nsurv == 32) {                                                            \
                    knn_refine<S>(ws, k, lane, 32);                                           \
                    nsurv = 0;                                                                \
                    RELOAD_G();                                                               \
                }                                                                             \
            }                                                                                 \
        }                                                                                     \
    }
            auto stream_table = [&](auto g0_tag) {
                constexpr bool G0 = decltype(g0_tag)::value;
                Blk ra, rb;
                load_block(ra, p.Xb, 0, lane);
                rb = ra;
#pragma unroll 1
                for (int t = 0; t < n_blocks; t += 2) {
                    if (t + 1 < n_blocks) load_block(rb, p.Xb, t + 1, lane);
                    FILTER_BLOCK(ra, t)
                    if (t + 1 < n_blocks) {
                        if (t + 2 < n_blocks) load_block(ra, p.Xb, t + 2, lane);
                        FILTER_BLOCK(rb, t + 1)
                    }
                }
            };
            // group 0 = lattice slots {}, {0}, {1}, {0,1}: when only {0,1} is asked for (the batch without
            // high features), the group is bounded by that slot's own sum (lattice_filter<true>)
            if ((SLOT(0) < 0) & (SLOT(1) < 0) & (SLOT(2) < 0)) stream_table(TrueTag{});
            else stream_table(FalseTag{});
#undef FILTER_BLOCK
            while (qtail > qhead) {
                const int r = knn_exact_test<S>(ws, lane, q, p.N, qhead, min(32, qtail - qhead), nsurv);
                qhead += r & 0xff;
                nsurv = r >> 8;
                if (nsurv == 32) {
                    knn_refine<S>(ws, k, lane, 32);
                    nsurv = 0;
                }
            }
            if (nsurv) knn_refine<S>(ws, k, lane, nsurv);
            knn_emit<S>(ws, p, q, lane);
            has_prev = true;
        }
    }
}

size_t knn_lattice_smem_bytes(int k, int warps) {
    return 128 + static_cast<size_t>(warps) * knn_warp_words(k) * 4;
}


cudaError_t knn_lattice_launch(const KnnParams& p, int grid, cudaStream_t stream) {
    const size_t smem = knn_lattice_smem_bytes(p.k, p.warps);
    const int stride = knn_list_stride(p.k);
    auto kernel = stride == 12 ? knn_lattice_kernel<12> : stride == 20 ? knn_lattice_kernel<20>
                  : stride == 28 ? knn_lattice_kernel<28> : knn_lattice_kernel<36>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kernel<<<grid, p.warps * 32, smem, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace snaps
