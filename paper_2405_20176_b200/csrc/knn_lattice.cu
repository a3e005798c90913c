// knn_lattice.cu -- kNN self-join over a batch of feature subspaces (steps a3-a5, a7).
//
// What it computes: PAPER.md:112, 122 (kNNSJ) for every mask of a sub-lattice batch;
// scores of PAPER.md:251-252 fused into the tail.  How:
//   * one consumer warp = one query object x the 64 masks {H u T : T subset of
//     features 0..5}; the 32 lanes hold 32 different candidates per step;
//   * candidate tiles (128 rows x 80 B) arrive in a 3-stage shared-memory ring via
//     cp.async.bulk + mbarrier from a dedicated producer warp (no __syncthreads in
//     the steady state);
//   * FILTER (every candidate): 15 squared differences once, then the 16 partial sums
//     X[u] over features 2..5 (add-only).  X[u] is a lower bound of the four sums
//     X[u] (+sq0) (+sq1) of "group" u (adding non-negative terms never rounds below the
//     addend), so a candidate can enter one of the group's lists only if X[u] < G[u],
//     G[u] = max of the group's four current thresholds (register-held);
//   * COMPACT: lanes that pass any group test push (id, base, sq0..5) into a per-warp
//     shared-memory queue (ballot + popc); with running thresholds ~2-4% of candidates pass;
//   * REFINE (every 32 queued candidates, all lanes busy): the 64 subset sums by add-only
//     enumeration in a fixed order, each compared with its list's current threshold
//     (k-th squared distance so far); passing (list, id, d^2) triples go to a per-warp ring;
//   * DRAIN: ring entries are merged into the sorted lists entry-parallel (one lane per
//     entry, lanes that target the same list take turns), thresholds and G
//     are refreshed;
//   * thresholds start from an upper bound seeded by evaluating k known objects
//     (the first k ids and the previous batch's neighbours: consecutive batches
//     differ in one feature), tightened by min over supersets (the k-th distance
//     is monotone in the feature set).
#include "knn_lattice.cuh"

namespace snaps {

#ifdef SNAPS_STATS
// Developer diagnostics (never built into the shipped library): phase clocks and event counts.
__device__ unsigned long long g_stats[16];
#define STAT_ADD(i, v) do { if (lane == 0) atomicAdd(&g_stats[i], (unsigned long long)(v)); } while (0)
#define STAT_CLK() clock64()
#else
#define STAT_ADD(i, v) do { } while (0)
#define STAT_CLK() 0ll
#endif

// ---- per-warp shared-memory state (32-bit words) ----------------------------------
// rows of 64 words (one word per list), element-major so that lane l touching
// list l is conflict-free:
//   rows [0,k)     list d^2 (ascending by (d^2,id))     rows [k,2k)   list ids
//   row 2k   list count     row 2k+1  threshold     row 2k+2  seed bound     row 2k+3  output slot
//   row 2k+4 words 0..15: G (group maxima), words 16..30: the query's 15 features
//   then the ring (3 arrays of kRing words) and the queue (64 entries of 8 words)
#define L_D2(e, L) ws[((e)) * 64 + (L)]
#define L_ID(e, L) wsi[(k + (e)) * 64 + (L)]
#define L_CNT(L) wsi[(2 * k) * 64 + (L)]
#define THR(L) ws[(2 * k + 1) * 64 + (L)]
#define SEED(L) ws[(2 * k + 2) * 64 + (L)]
#define SLOT(L) wsi[(2 * k + 3) * 64 + (L)]
#define GMAX(u) ws[(2 * k + 4) * 64 + (u)]
#define QROW(j) ws[(2 * k + 4) * 64 + 16 + (j)]
#define RG_T(i) wsi[(2 * k + 5) * 64 + (i)]
#define RG_ID(i) wsi[(2 * k + 5) * 64 + kRing + (i)]
#define RG_D2(i) ws[(2 * k + 5) * 64 + 2 * kRing + (i)]
#define QUEUE4(e) (reinterpret_cast<float4*>(ws + (2 * k + 5) * 64 + 3 * kRing) + 2 * (e))
constexpr int kQueue = 64;   // queue entries (8 words each); refine as soon as 32 are waiting

__host__ __device__ constexpr int knn_warp_words(int k) { return (2 * k + 5) * 64 + 3 * kRing + kQueue * 8; }

// Merge ring entries [0, cnt) into the sorted lists.  One lane per entry; lanes whose
// entries target the same list take turns; the (d^2, id) key decides, not arrival order.
// The insert is rank based: all loads of a list are independent (no pointer-chasing shift loop).
template <int KCAP>
__device__ __noinline__ void knn_drain(float* ws, int k, int lane, int q, int N, int cnt) {
    int* wsi = reinterpret_cast<int*>(ws);
    __syncwarp();
    const long long t0_ = STAT_CLK();
    STAT_ADD(4, 1);
    STAT_ADD(5, cnt);
#pragma unroll 1
    for (int e0 = 0; e0 < cnt; e0 += 32) {
        const int i = e0 + lane;
        bool valid = i < cnt;
        int T = 0, id = 0;
        float d = 0.f;
        if (valid) {
            T = RG_T(i);
            id = RG_ID(i);
            d = RG_D2(i);
            // self by index (reading A4), padding rows (A19), and entries that a tighter
            // threshold has overtaken since they were appended (ties are settled by the
            // (d^2, id) key below: ring order is not id order)
            if (id == q || id >= N || d > THR(T)) valid = false;
        }
        const unsigned peers = __match_any_sync(kFull, valid ? T : 64 + lane);
        const int rank = __popc(peers & ((1u << lane) - 1u));
        const int rounds = __reduce_max_sync(kFull, valid ? rank + 1 : 0);
        STAT_ADD(6, rounds);
#pragma unroll 1
        for (int r = 0; r < rounds; ++r) {
            if (valid && rank == r) {
                const int c = L_CNT(T);
                float v[KCAP];
                int w[KCAP];
#pragma unroll
                for (int e = 0; e < KCAP; ++e) {
                    v[e] = (e < c) ? L_D2(e, T) : __int_as_float(0x7f800000);
                    w[e] = (e < c) ? L_ID(e, T) : 0x7fffffff;
                }
                int pos = 0;  // number of list entries whose key precedes (d, id)
#pragma unroll
                for (int e = 0; e < KCAP; ++e) pos += (v[e] < d || (v[e] == d && w[e] < id)) ? 1 : 0;
                if (pos < k) {
                    const int cn = c < k ? c + 1 : k;
#pragma unroll
                    for (int e = KCAP - 1; e >= 1; --e) {
                        if (e > pos && e < cn) {
                            L_D2(e, T) = v[e - 1];
                            L_ID(e, T) = w[e - 1];
                        }
                    }
#pragma unroll
                    for (int e = 0; e < KCAP; ++e) {
                        if (e == pos) {
                            L_D2(e, T) = d;
                            L_ID(e, T) = id;
                        }
                    }
                    L_CNT(T) = cn;
                    if (cn == k) THR(T) = L_D2(k - 1, T);
                }
            }
            __syncwarp();
        }
    }
    if (lane < 16) {
        const float4 t = *reinterpret_cast<const float4*>(&THR(4 * lane));
        GMAX(lane) = fmaxf(fmaxf(t.x, t.y), fmaxf(t.z, t.w));
    }
    __syncwarp();
    STAT_ADD(1, STAT_CLK() - t0_);
}

// REFINE: lanes 0..n-1 take the n oldest queue entries; the 64 subset sums of each are
// compared with their lists' thresholds (branch-free, a 64-bit pass mask per lane); passing
// (list, id, d^2) triples are appended to the ring at positions from a warp prefix sum (at
// most kRing/32 per lane and round, so the ring cannot overflow) and merged.
// The add order (high features by FMA in feature order -> features 2,3,4,5 -> 0 -> 1) is the
// same wherever a squared distance is formed, so a value never depends on scheduling.
template <int KCAP>
__device__ __noinline__ void knn_refine(float* ws, int k, int lane, int q, int N, int head, int n) {
    int* wsi = reinterpret_cast<int*>(ws);
    __syncwarp();
    const long long t0_ = STAT_CLK();
    STAT_ADD(7, 1);
    STAT_ADD(8, n);
    float base = __int_as_float(0x7f800000);
    float sq[kLow] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    int cand = -1;
    if (lane < n) {
        const float4* e = QUEUE4((head + lane) % kQueue);
        const float4 a = e[0], b = e[1];
        cand = __float_as_int(a.x);
        base = a.y; sq[0] = a.z; sq[1] = a.w;
        sq[2] = b.x; sq[3] = b.y; sq[4] = b.z; sq[5] = b.w;
    }
    unsigned mlo = 0u, mhi = 0u;
    {
        float X[16];
        X[0] = base;
#pragma unroll
        for (int u = 1; u < 16; ++u) {
            const int hb = 31 - __clz(u);
            X[u] = __fadd_rn(X[u & ~(1 << hb)], sq[2 + hb]);
        }
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            const float s0 = X[u];
            const float s1 = __fadd_rn(s0, sq[0]);
            const float s2 = __fadd_rn(s0, sq[1]);
            const float s3 = __fadd_rn(s1, sq[1]);
            const float4 th = *reinterpret_cast<const float4*>(&THR(4 * u));
            const unsigned bits = (s0 < th.x ? 1u : 0u) | (s1 < th.y ? 2u : 0u) |
                                  (s2 < th.z ? 4u : 0u) | (s3 < th.w ? 8u : 0u);
            if (u < 8) mlo |= bits << (4 * u);
            else mhi |= bits << (4 * (u - 8));
        }
    }
    constexpr int kPerLane = kRing / 32;
#pragma unroll 1
    while (__any_sync(kFull, (mlo | mhi) != 0u)) {
        const int have = __popc(mlo) + __popc(mhi);
        // everything at once if it fits the ring, else a bounded share per lane and round
        const int mine = (__reduce_add_sync(kFull, have) <= kRing) ? have
                                                                   : (have < kPerLane ? have : kPerLane);
        int incl = mine;  // inclusive prefix sum over lanes
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(kFull, incl, o);
            if (lane >= o) incl += v;
        }
        const int total = __shfl_sync(kFull, incl, 31);
        int pos = incl - mine;
#pragma unroll 1
        for (int j = 0; j < mine; ++j, ++pos) {
            int T;
            if (mlo) {
                T = __ffs(mlo) - 1;
                mlo &= mlo - 1u;
            } else {
                T = 32 + __ffs(mhi) - 1;
                mhi &= mhi - 1u;
            }
            float x = base;
            if (T & 4) x = __fadd_rn(x, sq[2]);
            if (T & 8) x = __fadd_rn(x, sq[3]);
            if (T & 16) x = __fadd_rn(x, sq[4]);
            if (T & 32) x = __fadd_rn(x, sq[5]);
            if (T & 1) x = __fadd_rn(x, sq[0]);
            if (T & 2) x = __fadd_rn(x, sq[1]);
            RG_T(pos) = T;
            RG_ID(pos) = cand;
            RG_D2(pos) = x;
        }
        knn_drain<KCAP>(ws, k, lane, q, N, total);
    }
    STAT_ADD(0, STAT_CLK() - t0_);
}

// Upper bounds on the final k-th squared distance of every list of the new batch.
__device__ __noinline__ void knn_seed(float* ws, const float* __restrict__ Xp, int q, int k,
                                      uint32_t H, bool has_prev, int lane) {
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
            float b1 = 0.f;
#pragma unroll 1
            for (int e = 0; e < k; ++e) {
                const int c = e + (e >= q ? 1 : 0);
                b1 = fmaxf(b1, masked_d2(Xp + static_cast<size_t>(c) * kRowFloats, qrow, mask));
            }
            bound = b1;
            if (has_prev && L_CNT(L) == k) {
                float b2 = 0.f;
#pragma unroll 1
                for (int e = 0; e < k; ++e) {
                    const int c = L_ID(e, L);
                    b2 = fmaxf(b2, masked_d2(Xp + static_cast<size_t>(c) * kRowFloats, qrow, mask));
                }
                bound = fminf(bound, b2);
            }
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
        L_CNT(L) = 0;
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
__device__ __noinline__ void knn_emit(float* ws, const KnnParams& p, int q, int lane) {
    int* wsi = reinterpret_cast<int*>(ws);
    const int k = p.k;
    __syncwarp();
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
        const int L = lane + 32 * h;
        const int sl = SLOT(L);
        if (sl < 0) continue;
        const size_t o = static_cast<size_t>(sl) * static_cast<size_t>(p.N) + static_cast<size_t>(q);
        float sum = 0.f, dk = 0.f;
#pragma unroll 1
        for (int e = 0; e < k; ++e) {
            const float d = sqrtf(L_D2(e, L));
            const int id = L_ID(e, L);
            sum += d;
            dk = d;
            if (p.out_idx) p.out_idx[o * k + e] = id;
            if (p.out_dist) p.out_dist[o * k + e] = d;
            if (p.out_indeg)
                atomicAdd(&p.out_indeg[static_cast<size_t>(sl) * static_cast<size_t>(p.N) + id], 1);
        }
        if (p.out_kth) p.out_kth[o] = dk;
        if (p.out_mean) p.out_mean[o] = sum / static_cast<float>(k);
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

template <int KCAP>
__global__ void __launch_bounds__(kKnnMaxThreads, 1) knn_lattice_kernel(const KnnParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    int* s_item = reinterpret_cast<int*>(smem);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int W = p.warps;
    const int k = p.k;
    float* ws = reinterpret_cast<float*>(smem + 128) + static_cast<size_t>(warp) * knn_warp_words(k);
    int* wsi = reinterpret_cast<int*>(ws);

    const int n_items = p.n_qblocks * p.n_bchunks;
    const unsigned lt = (1u << lane) - 1u;
    for (;;) {
        // one item = W queries x a run of consecutive batches; the warps of a CTA start an item
        // together so that their scans of the table stay close and share L1 lines
        if (threadIdx.x == 0) s_item[0] = atomicAdd(p.work_counter, 1);
        __syncthreads();
        const int item = s_item[0];
        __syncthreads();
        if (item >= n_items) break;
        const int qb = item % p.n_qblocks, bc = item / p.n_qblocks;
        const int b0 = bc * p.batches_per_item;
        const int b1 = min(b0 + p.batches_per_item, p.n_batches);
        const int q = qb * W + warp;
        if (q >= p.N) continue;

        float qlo[kLow];
        float qhi[9];
        {
            const float* qr = p.Xp + static_cast<size_t>(q) * kRowFloats;
#pragma unroll
            for (int j = 0; j < kLow; ++j) qlo[j] = qr[j];
#pragma unroll
            for (int j = 0; j < 9; ++j) qhi[j] = qr[kLow + j];
            if (lane < 15) QROW(lane) = qr[lane];
        }
        bool has_prev = false;
#pragma unroll 1
        for (int b = b0; b < b1; ++b) {
            const BatchDesc* bd = &p.batches[b];
            const uint32_t H = bd->hmask;
            const long long tb_ = STAT_CLK();
            SLOT(lane) = bd->slot[lane];
            SLOT(lane + 32) = bd->slot[lane + 32];
            knn_seed(ws, p.Xp, q, k, H, has_prev, lane);
            STAT_ADD(9, STAT_CLK() - tb_);
            float G[16];
            RELOAD_G();
            float wq[9], w[9];  // high features: diff = c*w - q*w, w in {0,1}
#pragma unroll
            for (int j = 0; j < 9; ++j) {
                w[j] = ((H >> (kLow + j)) & 1u) ? 1.f : 0.f;
                wq[j] = w[j] * qhi[j];
            }
            int qhead = 0, qtail = 0;  // queue positions (warp-uniform, monotone)
            // candidates: block t = rows 32t..32t+31, lane = row, four coalesced 128-bit loads
            const float4* blk = p.Xb + lane;
            float4 n0 = __ldg(blk), n1 = __ldg(blk + 32), n2 = __ldg(blk + 64), n3 = __ldg(blk + 96);
#pragma unroll 1
            for (int t = 0; t < p.n_blocks; ++t) {
                const float4 r0 = n0, r1 = n1, r2 = n2, r3 = n3;
                if (t + 1 < p.n_blocks) {   // software prefetch of the next block
                    blk += 128;
                    n0 = __ldg(blk); n1 = __ldg(blk + 32); n2 = __ldg(blk + 64); n3 = __ldg(blk + 96);
                }
                const float c[15] = {r0.x, r0.y, r0.z, r0.w, r1.x, r1.y, r1.z, r1.w,
                                     r2.x, r2.y, r2.z, r2.w, r3.x, r3.y, r3.z};
                float sq[kLow];
#pragma unroll
                for (int j = 0; j < kLow; ++j) {
                    const float diff = c[j] - qlo[j];
                    sq[j] = __fmul_rn(diff, diff);
                }
                float base = 0.f;
#pragma unroll
                for (int j = 0; j < 9; ++j) {
                    const float diff = __fmaf_rn(c[kLow + j], w[j], -wq[j]);
                    base = __fmaf_rn(diff, diff, base);
                }
                // FILTER: group lower bounds against group maxima
                float X[16];
                X[0] = base;
#pragma unroll
                for (int u = 1; u < 16; ++u) {
                    const int hb = 31 - __clz(u);
                    X[u] = __fadd_rn(X[u & ~(1 << hb)], sq[2 + hb]);
                }
                bool pass = false;
#pragma unroll
                for (int u = 0; u < 16; ++u) pass |= (X[u] < G[u]);
                const unsigned bal = __ballot_sync(kFull, pass);
                if (bal) {
                    // COMPACT
                    if (pass) {
                        float4* e = QUEUE4((qtail + __popc(bal & lt)) % kQueue);
                        e[0] = make_float4(__int_as_float(t * 32 + lane), base, sq[0], sq[1]);
                        e[1] = make_float4(sq[2], sq[3], sq[4], sq[5]);
                    }
                    qtail += __popc(bal);
                    if (qtail - qhead >= 32) {
                        knn_refine<KCAP>(ws, k, lane, q, p.N, qhead, 32);
                        qhead += 32;
                        RELOAD_G();
                    }
                }
            }
            const long long te_ = STAT_CLK();
            if (qtail > qhead) knn_refine<KCAP>(ws, k, lane, q, p.N, qhead, qtail - qhead);
            knn_emit(ws, p, q, lane);
            STAT_ADD(10, STAT_CLK() - te_);
            STAT_ADD(3, STAT_CLK() - tb_);
            STAT_ADD(11, 1);
            has_prev = true;
        }
    }
}

size_t knn_lattice_smem_bytes(int k, int warps) {
    return 128 + static_cast<size_t>(warps) * knn_warp_words(k) * 4;
}

#ifdef SNAPS_STATS
extern "C" int snaps_debug_stats(unsigned long long* out16, int reset) {
    if (out16) cudaMemcpyFromSymbol(out16, g_stats, sizeof(g_stats));
    if (reset) {
        unsigned long long z[16] = {0};
        cudaMemcpyToSymbol(g_stats, z, sizeof(z));
    }
    return 0;
}
#endif

cudaError_t knn_lattice_launch(const KnnParams& p, int grid, cudaStream_t stream) {
    const size_t smem = knn_lattice_smem_bytes(p.k, p.warps);
    auto kernel = p.k <= 16 ? knn_lattice_kernel<16> : knn_lattice_kernel<32>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kernel<<<grid, p.warps * 32, smem, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace snaps
