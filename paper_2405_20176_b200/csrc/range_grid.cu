// range_grid.cu -- DSSJ for a whole grid of radii in one scan (NEXT-1, Fig. 3):
// the result set of eps_max contains the result sets of every smaller eps_j, so the join runs once
// at eps_max and each neighbour is binned by the smallest grid radius that contains it; cumulative
// sums over the bins give the count and the distance sum for every eps_j.
// Same filter / compact / exact test / refine structure as range_lattice.cu (the exact test is
// against the largest radius of every list); the list owner keeps a per-radius histogram
// (count, sum of distances) in shared memory.
#include "range_grid.cuh"

namespace snaps {

constexpr int kGQueue = 64;

// per-warp shared-memory words; G = number of radii (runtime)
//   SLOT[64] | QROW[16] | MT 32x36 | queue 64x8 | TMAX[64] | THR[64][G] | HCNT[64][G] | HSUM[64][G]
#define G_SLOT(L) wsi[(L)]
#define G_MT(T, j) ws[80 + (T) * 36 + (j)]
#define G_QUEUE4 (reinterpret_cast<float4*>(ws + 80 + 32 * 36))
// survivors of the exact test (at most 32): taken into registers before the transpose is written
#define G_SURV4 (reinterpret_cast<float4*>(&G_MT(0, 0)))
#define G_TMAX(L) ws[80 + 32 * 36 + kGQueue * 8 + (L)]   // the largest radius of list L (-1: unused slot)
#define G_BASE (80 + 32 * 36 + kGQueue * 8 + 64)
#define G_THR(L, g) ws[G_BASE + (L) * G + (g)]
#define G_HCNT(L, g) wsi[G_BASE + 64 * G + (L) * G + (g)]
#define G_HSUM(L, g) ws[G_BASE + 128 * G + (L) * G + (g)]

__host__ __device__ inline int range_grid_warp_words(int G) { return G_BASE + 192 * G; }

// self by index (A4) and padding rows (A19) get an infinite base when they leave the queue
__device__ __noinline__ int range_grid_exact_test(float* ws, int lane, int q, int N, int head, int n, int nb) {
    __syncwarp();
    return lattice_exact_test(G_QUEUE4, kGQueue, G_SURV4, &G_TMAX(0), lane, q, N, head, n, nb);
}

__device__ __noinline__ void range_grid_refine(float* ws, int G, bool with_sum, int lane, int n) {
    int* wsi = reinterpret_cast<int*>(ws);
    __syncwarp();
    PairTerms pt;
    survivors_pop(G_SURV4, lane, n, pt);
    __syncwarp();   // the transpose overwrites the survivors' storage
    float X8[8];
    lattice_partial8(pt, X8);
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        lattice_sums_to_transpose(pt, X8, half, &G_MT(0, 0), lane);
        __syncwarp();
        const int T = 32 * half + lane;
        const float thr = G_TMAX(T);
        // A neighbour's bin = the smallest radius that contains it (radii ascend).  The bin is guessed from the
        // distance itself, as if the list's radii were evenly spaced between the smallest and the largest (the
        // library's own grids are, reading A22), and the guess is settled against the exact thresholds on
        // either side: one shared-memory round trip per neighbour when the guess is right, any grid stays exact.
        const float t_first = G_THR(T, 0);
        const float e_first = sqrtf(fmaxf(t_first, 0.f)), e_last = sqrtf(fmaxf(thr, 0.f));
        const float per_eps = (G > 1 && e_last > e_first) ? static_cast<float>(G - 1) / (e_last - e_first) : 0.f;
        unsigned mask = 0u;
#pragma unroll
        for (int j4 = 0; j4 < 8; ++j4) {
            const float4 m = *reinterpret_cast<const float4*>(&G_MT(lane, 4 * j4));
            mask |= (m.x < thr ? 1u : 0u) << (4 * j4);
            mask |= (m.y < thr ? 1u : 0u) << (4 * j4 + 1);
            mask |= (m.z < thr ? 1u : 0u) << (4 * j4 + 2);
            mask |= (m.w < thr ? 1u : 0u) << (4 * j4 + 3);
        }
        // bin of one neighbour: guess, then settle against the exact thresholds on either side
        auto bin_of = [&](float d2, float dd) -> int {
            int g = min(max(__float2int_ru((dd - e_first) * per_eps), 0), G - 1);
            const float below = g > 0 ? G_THR(T, g - 1) : -1.f, here = G_THR(T, g);
            if (d2 < below) {
                --g;
                while (g > 0 && d2 < G_THR(T, g - 1)) --g;
            } else if (!(d2 < here)) {
                ++g;
                while (!(d2 < G_THR(T, g))) ++g;             // ends: d2 < the largest threshold
            }
            return g;
        };
        // two neighbours per trip: their bin searches and histogram reads overlap; the updates keep candidate order
#pragma unroll 1
        while (mask) {
            const int j0 = __ffs(mask) - 1;
            mask &= mask - 1u;
            const bool two = mask != 0u;
            const int j1 = two ? __ffs(mask) - 1 : j0;
            if (two) mask &= mask - 1u;
            const float d2a = G_MT(lane, j0), d2b = G_MT(lane, j1);
            const float dda = sqrtf(d2a), ddb = sqrtf(d2b);
            const int ga = bin_of(d2a, dda), gb = bin_of(d2b, ddb);
            const int ca = G_HCNT(T, ga), cb = G_HCNT(T, gb);
            const float sa = with_sum ? G_HSUM(T, ga) : 0.f, sb = with_sum ? G_HSUM(T, gb) : 0.f;
            if (two && ga == gb) {
                G_HCNT(T, ga) = ca + 2;
                if (with_sum) G_HSUM(T, ga) = (sa + dda) + ddb;
            } else {
                G_HCNT(T, ga) = ca + 1;
                if (with_sum) G_HSUM(T, ga) = sa + dda;
                if (two) {
                    G_HCNT(T, gb) = cb + 1;
                    if (with_sum) G_HSUM(T, gb) = sb + ddb;
                }
            }
        }
        __syncwarp();
    }
}

__global__ void __launch_bounds__(kRangeGridMaxThreads, 1) range_grid_kernel(const RangeGridParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int G = p.G;
    float* ws = reinterpret_cast<float*>(smem) + static_cast<size_t>(warp) * range_grid_warp_words(G);
    int* wsi = reinterpret_cast<int*>(ws);
    const bool with_sum = p.out_sum != nullptr || p.out_mean != nullptr;
    const long long n_items = static_cast<long long>(p.nq) * p.n_batches;
    const unsigned lt = (1u << lane) - 1u;
    const int n_blocks = p.n_blocks;
    for (;;) {
        long long item = 0;
        if (lane == 0) item = atomicAdd(p.work_counter, 1ull);
        item = __shfl_sync(kFull, item, 0);
        if (item >= n_items) break;
        const int q = p.q_begin + static_cast<int>(item % p.nq);
        const int b = static_cast<int>(item / p.nq);
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
        const BatchDesc* bd = &p.batches[b];
        const uint32_t H = bd->hmask;
        __syncwarp();
        for (int h = 0; h < 2; ++h) {
            const int L = lane + 32 * h;
            const int sl = bd->slot[L];
            G_SLOT(L) = sl;
            for (int g = 0; g < G; ++g) {
                G_THR(L, g) = sl >= 0 ? p.thr_grid[static_cast<size_t>(sl) * G + g] : -1.f;
                G_HCNT(L, g) = 0;
                G_HSUM(L, g) = 0.f;
            }
            G_TMAX(L) = G_THR(L, G - 1);
        }
        __syncwarp();
        filter_query_init(fq, qhi, H);
        const bool g0_both = (G_SLOT(0) < 0) & (G_SLOT(1) < 0) & (G_SLOT(2) < 0);
        float Gm[16];
#pragma unroll
        for (int u = 0; u < 16; ++u)
            Gm[u] = fmaxf(fmaxf(G_TMAX(4 * u), G_TMAX(4 * u + 1)), fmaxf(G_TMAX(4 * u + 2), G_TMAX(4 * u + 3)));
        int qhead = 0, qtail = 0, nsurv = 0;
        Blk nx;
        load_block(nx, p.Xb, 0, lane);
#pragma unroll 1
        for (int t = 0; t < n_blocks; ++t) {
            const Blk r = nx;
            if (t + 1 < n_blocks) load_block(nx, p.Xb, t + 1, lane);
            PairTerms pt;
            const bool pass = g0_both ? lattice_filter<true>(r, fq, Gm, pt) : lattice_filter<false>(r, fq, Gm, pt);
            const unsigned bal = __ballot_sync(kFull, pass);
            if (bal) {
                qtail += queue_push(G_QUEUE4, kGQueue, qtail, pass, bal, lt, t * 32 + lane, pt);
                while (qtail - qhead >= 32) {
                    const int r_ = range_grid_exact_test(ws, lane, q, p.N, qhead, 32, nsurv);
                    qhead += r_ & 0xff;
                    nsurv = r_ >> 8;
                    if (nsurv == 32) {
                        range_grid_refine(ws, G, with_sum, lane, 32);
                        nsurv = 0;
                    }
                }
            }
        }
        while (qtail > qhead) {
            const int r_ = range_grid_exact_test(ws, lane, q, p.N, qhead, min(32, qtail - qhead), nsurv);
            qhead += r_ & 0xff;
            nsurv = r_ >> 8;
            if (nsurv == 32) {
                range_grid_refine(ws, G, with_sum, lane, 32);
                nsurv = 0;
            }
        }
        if (nsurv) range_grid_refine(ws, G, with_sum, lane, nsurv);
        // cumulative over the radii: count(eps_g) = sum of the bins <= g
        __syncwarp();
        for (int h = 0; h < 2; ++h) {
            const int L = lane + 32 * h;
            const int sl = G_SLOT(L);
            if (sl < 0) continue;
            int cnt = 0;
            float tot = 0.f;
            for (int g = 0; g < G; ++g) {
                cnt += G_HCNT(L, g);
                tot += G_HSUM(L, g);
                const size_t o = (static_cast<size_t>(sl) * G + g) * static_cast<size_t>(p.nq) + (q - p.q_begin);
                p.out_count[o] = static_cast<uint32_t>(cnt);
                if (p.out_sum) p.out_sum[o] = tot;
                if (p.out_mean) p.out_mean[o] = cnt > 0 ? tot / static_cast<float>(cnt) : 0.f;
            }
        }
    }
}

size_t range_grid_smem_bytes(int G, int warps) { return static_cast<size_t>(warps) * range_grid_warp_words(G) * 4; }

cudaError_t range_grid_launch(const RangeGridParams& p, int grid, cudaStream_t stream) {
    const size_t smem = range_grid_smem_bytes(p.G, p.warps);
    cudaError_t e = cudaFuncSetAttribute(range_grid_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    range_grid_kernel<<<grid, p.warps * 32, smem, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace snaps
