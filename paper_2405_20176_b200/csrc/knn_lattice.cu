// knn_lattice.cu -- kNN self-join over a batch of feature subspaces (steps a3-a5, a7).
//
// What it computes: PAPER.md:112, 122 (kNNSJ) for every mask of a sub-lattice batch;
// scores of PAPER.md:251-252 fused into the tail.  How:
//   * one consumer warp = one query object x the 64 masks {H u T : T subset of
//     features 0..5}; the 32 lanes hold 32 different candidates per step;
//   * candidate tiles (128 rows x 80 B) arrive in a 3-stage shared-memory ring via
//     cp.async.bulk + mbarrier from a dedicated producer warp (no __syncthreads in
//     the steady state);
//   * per (lane = candidate): 15 squared differences once, then the 64 subset sums
//     by add-only enumeration (63 FADDs), each compared with a register-held
//     threshold (current k-th squared distance of that (query, mask) list);
//   * a warp vote per group of 4 sums gates the rare path: passing candidates are
//     appended to a small per-list pending buffer in shared memory; buffers are
//     merged into the sorted lists lane-parallel (one lane per list) and the
//     thresholds re-read;
//   * thresholds start from an upper bound seeded by evaluating k known objects
//     (the first k ids and the previous batch's neighbours: consecutive batches
//     differ in one feature), tightened by min over supersets (the k-th distance
//     is monotone in the feature set).
#include "knn_lattice.cuh"

namespace snaps {

// ---- per-warp shared-memory state -------------------------------------------------
// rows of 64 words (one word per list), element-major so that lane l touching
// list l is conflict-free:
//   [0,k)        list d^2 (ascending by (d^2,id))     [k,2k)           list ids
//   [2k,2k+P)    pending d^2                          [2k+P,2k+2P)     pending ids
//   then rows: pending count, list count, threshold, seed bound, output slot, query row
#define L_D2(e, L) ws[((e)) * 64 + (L)]
#define L_ID(e, L) wsi[(k + (e)) * 64 + (L)]
#define P_D2(s, L) ws[(2 * k + (s)) * 64 + (L)]
#define P_ID(s, L) wsi[(2 * k + kPend + (s)) * 64 + (L)]
#define P_CNT(L) wsi[(2 * k + 2 * kPend) * 64 + (L)]
#define L_CNT(L) wsi[(2 * k + 2 * kPend + 1) * 64 + (L)]
#define THR(L) ws[(2 * k + 2 * kPend + 2) * 64 + (L)]
#define SEED(L) ws[(2 * k + 2 * kPend + 3) * 64 + (L)]
#define SLOT(L) wsi[(2 * k + 2 * kPend + 4) * 64 + (L)]
#define QROW(j) ws[(2 * k + 2 * kPend + 5) * 64 + (j)]

// Merge every list's pending entries into its sorted list; lane l owns lists l, l+32.
__device__ __noinline__ void knn_drain(float* ws, int k, int lane) {
    int* wsi = reinterpret_cast<int*>(ws);
    __syncwarp();
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
        const int L = lane + 32 * h;
        int n = P_CNT(L);
        if (n == 0) continue;
        n = n < kPend ? n : kPend;
        int c = L_CNT(L);
#pragma unroll 1
        for (int e = 0; e < n; ++e) {
            const float d = P_D2(e, L);
            const int id = P_ID(e, L);
            int pos;
            if (c == k) {
                const float ld = L_D2(k - 1, L);
                const int li = L_ID(k - 1, L);
                if (!(d < ld || (d == ld && id < li))) continue;
                pos = k - 1;
            } else {
                pos = c++;
            }
            while (pos > 0) {
                const float pd = L_D2(pos - 1, L);
                const int pi = L_ID(pos - 1, L);
                if (pd < d || (pd == d && pi < id)) break;
                L_D2(pos, L) = pd;
                L_ID(pos, L) = pi;
                --pos;
            }
            L_D2(pos, L) = d;
            L_ID(pos, L) = id;
        }
        L_CNT(L) = c;
        P_CNT(L) = 0;
        THR(L) = (c == k) ? L_D2(k - 1, L) : SEED(L);
    }
    __syncwarp();
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
        P_CNT(L) = 0;
        L_CNT(L) = 0;
        THR(L) = SEED(L);
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

#define RELOAD_THR()                                                          \
    do {                                                                      \
        const float4* t4 = reinterpret_cast<const float4*>(&THR(0));          \
        _Pragma("unroll") for (int i4 = 0; i4 < 16; ++i4) {                   \
            const float4 v = t4[i4];                                          \
            thr[4 * i4 + 0] = v.x;                                            \
            thr[4 * i4 + 1] = v.y;                                            \
            thr[4 * i4 + 2] = v.z;                                            \
            thr[4 * i4 + 3] = v.w;                                            \
        }                                                                     \
    } while (0)

#define TRY_APPEND(bit, sval, Lidx)                                           \
    if (pend & (1u << (bit))) {                                               \
        const int slot_ = atomicAdd(&P_CNT(Lidx), 1);                         \
        if (slot_ < kPend) {                                                  \
            P_D2(slot_, Lidx) = (sval);                                       \
            P_ID(slot_, Lidx) = cand;                                         \
            pend &= ~(1u << (bit));                                           \
        }                                                                     \
        want |= (slot_ >= kPend / 2 - 1);                                     \
    }

// Rare path after a candidate step: merge pending entries, then retry the appends that
// found their list's pending buffer full.  The squared distance is re-derived in the
// exact operation order of the main loop, so the value does not depend on which lane
// overflowed.
__device__ __noinline__ void knn_fix(float* ws, int k, int lane, unsigned long long ovf,
                                     const float* __restrict__ crow, uint32_t H, int cand) {
    int* wsi = reinterpret_cast<int*>(ws);
    knn_drain(ws, k, lane);
    while (__any_sync(kFull, ovf != 0ull)) {
        if (ovf != 0ull) {
            const int L = __ffsll(static_cast<long long>(ovf)) - 1;
            float base = 0.f;
#pragma unroll
            for (int j = 0; j < 9; ++j) {
                const float wj = ((H >> (kLow + j)) & 1u) ? 1.f : 0.f;
                const float diff = __fmaf_rn(crow[kLow + j], wj, -(wj * QROW(kLow + j)));
                base = __fmaf_rn(diff, diff, base);
            }
            float acc = base;
#pragma unroll
            for (int jj = 0; jj < kLow; ++jj) {
                const int j = (jj < 4) ? jj + 2 : jj - 4;  // order 2,3,4,5,0,1 as in the lattice walk
                const float diff = crow[j] - QROW(j);
                const float sq = __fmul_rn(diff, diff);
                if ((L >> j) & 1) acc = __fadd_rn(acc, sq);
            }
            bool done = true;
            if (acc < THR(L)) {
                const int slot_ = atomicAdd(&P_CNT(L), 1);
                if (slot_ < kPend) {
                    P_D2(slot_, L) = acc;
                    P_ID(slot_, L) = cand;
                } else {
                    done = false;
                }
            }
            if (done) ovf &= ~(1ull << L);
        }
        knn_drain(ws, k, lane);
    }
}

__global__ void __launch_bounds__(kKnnMaxThreads, 1) knn_lattice_kernel(const KnnParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    float* tiles = reinterpret_cast<float*>(smem);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + kStages * kTileBytes);
    uint64_t* empty = full + kStages;
    int* s_item = reinterpret_cast<int*>(empty + kStages);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int W = p.warps;
    const int k = p.k;
    const int ws_floats = (2 * k + 2 * kPend + 6) * 64;
    float* ws = reinterpret_cast<float*>(smem + kStages * kTileBytes + 128) +
                static_cast<size_t>(warp < W ? warp : 0) * ws_floats;
    int* wsi = reinterpret_cast<int*>(ws);

    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], W);
        }
        mbar_fence_init();
    }
    __syncthreads();

    uint32_t g = 0;  // tiles consumed so far by this CTA (same value in every warp)
    const int n_items = p.n_qblocks * p.n_bchunks;
    for (;;) {
        if (threadIdx.x == 0) s_item[0] = atomicAdd(p.work_counter, 1);
        __syncthreads();
        const int item = s_item[0];
        __syncthreads();
        if (item >= n_items) break;
        const int qb = item % p.n_qblocks, bc = item / p.n_qblocks;
        const int b0 = bc * p.batches_per_item;
        const int b1 = min(b0 + p.batches_per_item, p.n_batches);
        const uint32_t ntile_total = static_cast<uint32_t>(b1 - b0) * p.n_tiles;

        if (warp == W) {
            // ---------------- producer warp: stream the whole table once per batch
            if (lane == 0) {
                for (uint32_t t = 0; t < ntile_total; ++t) {
                    const uint32_t gg = g + t;
                    const int s = gg % kStages;
                    const uint32_t ph = (gg / kStages) & 1u;
                    mbar_wait(&empty[s], ph ^ 1u);
                    mbar_arrive_expect_tx(&full[s], kTileBytes);
                    bulk_g2s(tiles + static_cast<size_t>(s) * kTileRows * kRowFloats,
                             p.Xp + static_cast<size_t>(t % p.n_tiles) * kTileRows * kRowFloats,
                             kTileBytes, &full[s]);
                }
            }
            g += ntile_total;
            __syncwarp();
            continue;
        }

        // ---------------- consumer warp: one query, all batches of this item
        const int q = qb * W + warp;
        const bool active = q < p.N;
        float qlo[kLow];
        float qhi[9];
        {
            const float* qr = p.Xp + static_cast<size_t>(active ? q : 0) * kRowFloats;
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
            if (active) {
                SLOT(lane) = bd->slot[lane];
                SLOT(lane + 32) = bd->slot[lane + 32];
                knn_seed(ws, p.Xp, q, k, H, has_prev, lane);
            }
            float thr[kLat];
            RELOAD_THR();
            float wq[9], w[9];  // high features: diff = c*w - q*w, w in {0,1}
#pragma unroll
            for (int j = 0; j < 9; ++j) {
                w[j] = ((H >> (kLow + j)) & 1u) ? 1.f : 0.f;
                wq[j] = w[j] * qhi[j];
            }
#pragma unroll 1
            for (int t = 0; t < p.n_tiles; ++t, ++g) {
                const int s = g % kStages;
                mbar_wait(&full[s], (g / kStages) & 1u);
                if (active) {
                    const float* tile = tiles + static_cast<size_t>(s) * kTileRows * kRowFloats;
#pragma unroll 1
                    for (int it = 0; it < kTileRows / 32; ++it) {
                        const int cand = t * kTileRows + it * 32 + lane;
                        const float4* row =
                            reinterpret_cast<const float4*>(tile + (it * 32 + lane) * kRowFloats);
                        const float4 r0 = row[0], r1 = row[1], r2 = row[2], r3 = row[3];
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
                        // padding rows and the query itself never enter a list (readings A4, A19)
                        if (cand >= p.N || cand == q) base = __int_as_float(0x7f800000);
                        unsigned long long ovf = 0ull;
                        bool want = false, touched = false;
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
                            const bool hit = (s0 < thr[4 * u]) | (s1 < thr[4 * u + 1]) |
                                             (s2 < thr[4 * u + 2]) | (s3 < thr[4 * u + 3]);
                            if (__any_sync(kFull, hit)) {
                                unsigned pend = (s0 < thr[4 * u] ? 1u : 0u) |
                                                (s1 < thr[4 * u + 1] ? 2u : 0u) |
                                                (s2 < thr[4 * u + 2] ? 4u : 0u) |
                                                (s3 < thr[4 * u + 3] ? 8u : 0u);
                                TRY_APPEND(0, s0, 4 * u + 0)
                                TRY_APPEND(1, s1, 4 * u + 1)
                                TRY_APPEND(2, s2, 4 * u + 2)
                                TRY_APPEND(3, s3, 4 * u + 3)
                                ovf |= static_cast<unsigned long long>(pend) << (4 * u);
                                touched = true;
                            }
                        }
                        if (touched) {
                            if (__any_sync(kFull, want || ovf != 0ull)) {
                                knn_fix(ws, k, lane, ovf,
                                        tile + (it * 32 + lane) * kRowFloats, H, cand);
                                RELOAD_THR();
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[s]);
            }
            if (active) {
                knn_drain(ws, k, lane);
                knn_emit(ws, p, q, lane);
            }
            has_prev = true;
        }
    }
}

size_t knn_lattice_smem_bytes(int k, int warps) {
    return static_cast<size_t>(kStages) * kTileBytes + 128 +
           static_cast<size_t>(warps) * (2 * k + 2 * kPend + 6) * 64 * 4;
}

cudaError_t knn_lattice_launch(const KnnParams& p, int grid, cudaStream_t stream) {
    const size_t smem = knn_lattice_smem_bytes(p.k, p.warps);
    cudaError_t e = cudaFuncSetAttribute(knn_lattice_kernel,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    knn_lattice_kernel<<<grid, (p.warps + 1) * 32, smem, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace snaps
