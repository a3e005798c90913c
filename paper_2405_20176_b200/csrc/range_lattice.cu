// range_lattice.cu -- eps range self-join (DSSJ) over a batch of feature subspaces
// (steps a3, a4, a6, a7).
//
// What it computes: PAPER.md:111, 154-156: for every object i and mask S the number of
// objects j != i with D(i,j;S) <= eps_S and the sum of those D
// (PAPER.md:165).  Same structure as knn_lattice.cu:
//   * one warp = one query x the 64 masks {H u T : T subset of features 0..5}; lanes = candidates
//     streamed from the blocked table (L2 resident, coalesced 128-bit loads, register prefetch);
//   * FILTER: the 16 partial sums X[u] over features 2..5 are lower bounds of their group's four
//     sums, so a candidate can be an eps-neighbour in group u only if X[u] < G[u] = the group's
//     largest eps^2 (constants per batch, register-held);
//   * COMPACT passing candidates into a per-warp queue; EXACT TEST every 32 of them (lane = candidate:
//     the 64 subset sums against the 64 thresholds, snaps_device.cuh); REFINE every 32 candidates
//     that have a sum below a threshold: lane = candidate
//     forms the 64 subset sums (add-only, fixed order), a 32 x 32 shared-memory transpose hands
//     them to the list owners (lane = list), which count the sums below eps^2 with one popcount
//     and add sqrt(d^2) of the hits to the list's running sum in candidate order (deterministic;
//     each list is touched by one lane only -- no atomics are needed at all).
#include "range_lattice.cuh"

namespace snaps {

constexpr int kRQueue = 64;  // queue entries of 8 words; exact test as soon as 32 are waiting

// per-warp shared-memory words
#define R_THR(L) ws[(L)]
#define R_SLOT(L) wsi[64 + (L)]
#define R_CNT(L) wsi[128 + (L)]
#define R_SUM(L) ws[192 + (L)]
#define R_QROW(j) ws[256 + (j)]
#define R_MT(T, j) ws[272 + (T) * 36 + (j)]
#define R_QUEUE4 (reinterpret_cast<float4*>(ws + 272 + 32 * 36))
// survivors of the exact test (at most 32): taken into registers before the transpose is written
#define R_SURV4 (reinterpret_cast<float4*>(&R_MT(0, 0)))

__host__ __device__ constexpr int range_warp_words() { return 272 + 32 * 36 + kRQueue * 8; }

// self (A4) and padding rows (A19) get an infinite base when they leave the queue: they never count
__device__ __noinline__ int range_exact_test(float* ws, int lane, int q, int N, int head, int n, int nb) {
    __syncwarp();
    return lattice_exact_test(R_QUEUE4, kRQueue, R_SURV4, &R_THR(0), lane, q, N, head, n, nb);
}

template <bool WITH_SUM>
__device__ __noinline__ void range_refine(float* ws, int lane, int n) {
    int* wsi = reinterpret_cast<int*>(ws);
    __syncwarp();
    PairTerms pt;
    survivors_pop(R_SURV4, lane, n, pt);
    __syncwarp();   // the transpose overwrites the survivors' storage
    float X8[8];   // partial sums over features 2,3,4; feature 5 is added per half
    lattice_partial8(pt, X8);
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        lattice_sums_to_transpose(pt, X8, half, &R_MT(0, 0), lane);
        __syncwarp();
        // ---- lane = list T: d^2 < nextafter(eps^2)  <=>  D <= eps (closed ball, reading A2)
        const int T = 32 * half + lane;
        const float thr = R_THR(T);
        unsigned mask = 0u;
#pragma unroll
        for (int j4 = 0; j4 < 8; ++j4) {
            const float4 m = *reinterpret_cast<const float4*>(&R_MT(lane, 4 * j4));
            mask |= (m.x < thr ? 1u : 0u) << (4 * j4);
            mask |= (m.y < thr ? 1u : 0u) << (4 * j4 + 1);
            mask |= (m.z < thr ? 1u : 0u) << (4 * j4 + 2);
            mask |= (m.w < thr ? 1u : 0u) << (4 * j4 + 3);
        }
        if (mask) {
            R_CNT(T) += __popc(mask);
            if (WITH_SUM) {
                float s = R_SUM(T);
#pragma unroll 1
                while (mask) {
                    const int j = __ffs(mask) - 1;
                    mask &= mask - 1u;
                    s += sqrtf(R_MT(lane, j));
                }
                R_SUM(T) = s;
            }
        }
        __syncwarp();
    }
}

template <bool WITH_SUM>
__global__ void __launch_bounds__(kRangeMaxThreads, 1) range_lattice_kernel(const RangeParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float* ws = reinterpret_cast<float*>(smem) + static_cast<size_t>(warp) * range_warp_words();
    int* wsi = reinterpret_cast<int*>(ws);
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
        }
#pragma unroll 1
        for (int b = b0; b < b1; ++b) {
            const BatchDesc* bd = &p.batches[b];
            const uint32_t H = bd->hmask;
            __syncwarp();
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int L = lane + 32 * h;
                R_THR(L) = bd->thr[L];
                R_SLOT(L) = bd->slot[L];
                R_CNT(L) = 0;
                R_SUM(L) = 0.f;
            }
            __syncwarp();
            filter_query_init(fq, qhi, H);
            float G[16];   // group maxima of the (constant) thresholds
#pragma unroll
            for (int u = 0; u < 16; ++u) {
                const float4 t = *reinterpret_cast<const float4*>(&R_THR(4 * u));
                G[u] = fmaxf(fmaxf(t.x, t.y), fmaxf(t.z, t.w));
            }
            int qhead = 0, qtail = 0, nsurv = 0;
#define FILTER_BLOCK(r, t_)                                                                   \
    {                                                                                         \
        PairTerms pt;                                                                         \
        const bool pass = lattice_filter<G0>(r, fq, G, pt);                                   \
        const unsigned bal = __ballot_sync(kFull, pass);                                      \
        if (bal) {                                                                            \
            qtail += queue_push(R_QUEUE4, kRQueue, qtail, pass, bal, lt, (t_) * 32 + lane, pt); \
            while (qtail - qhead >= 32) {                                                     \
                const int r_ = range_exact_test(ws, lane, q, p.N, qhead, 32, nsurv);          \
                qhead += r_ & 0xff;                                                           \
                nsurv = r_ >> 8;                                                              \
                if (nsurv == 32) {                                                            \
                    range_refine<WITH_SUM>(ws, lane, 32);                                     \
                    nsurv = 0;                                                                \
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
            // group 0 = lattice slots {}, {0}, {1}, {0,1}: when only {0,1} is asked for, the group is
            // bounded by that slot's own sum (X[0] alone is 0 when H is empty)
            if ((R_SLOT(0) < 0) & (R_SLOT(1) < 0) & (R_SLOT(2) < 0)) stream_table(TrueTag{});
            else stream_table(FalseTag{});
#undef FILTER_BLOCK
            while (qtail > qhead) {
                const int r = range_exact_test(ws, lane, q, p.N, qhead, min(32, qtail - qhead), nsurv);
                qhead += r & 0xff;
                nsurv = r >> 8;
                if (nsurv == 32) {
                    range_refine<WITH_SUM>(ws, lane, 32);
                    nsurv = 0;
                }
            }
            if (nsurv) range_refine<WITH_SUM>(ws, lane, nsurv);
            // ---- a7: counts, sums, means (0 when there is no neighbour: PAPER.md:266, reading A6)
            __syncwarp();
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int L = lane + 32 * h;
                const int sl = R_SLOT(L);
                if (sl < 0) continue;
                const size_t o = static_cast<size_t>(sl) * static_cast<size_t>(p.nq) + (q - p.q_begin);
                const int cnt = R_CNT(L);
                p.out_count[o] = static_cast<uint32_t>(cnt);
                if (WITH_SUM) {
                    const float tot = R_SUM(L);
                    if (p.out_sum) p.out_sum[o] = tot;
                    if (p.out_mean) p.out_mean[o] = cnt > 0 ? tot / static_cast<float>(cnt) : 0.f;
                }
            }
        }
    }
}

size_t range_lattice_smem_bytes(int warps) { return static_cast<size_t>(warps) * range_warp_words() * 4; }

cudaError_t range_lattice_launch(const RangeParams& p, int grid, cudaStream_t stream) {
    const bool with_sum = p.out_sum != nullptr || p.out_mean != nullptr;
    const size_t smem = range_lattice_smem_bytes(p.warps);
    auto kernel = with_sum ? range_lattice_kernel<true> : range_lattice_kernel<false>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kernel<<<grid, p.warps * 32, smem, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace snaps
