// range_grid.cu -- DSSJ for a whole grid of radii in one scan (NEXT-1, Fig. 3):
// the result set of eps_max contains the result sets of every smaller eps_j, so the join runs once
// at eps_max and each neighbour is binned by the smallest grid radius that contains it; cumulative
// sums over the bins give the count and the distance sum for every eps_j.
// Same filter / compact / refine structure as range_lattice.cu; the list owner keeps a
// per-radius histogram (count, sum of distances) in shared memory.
#include "range_grid.cuh"

namespace snaps {

constexpr int kGQueue = 64;
constexpr float kGInf = __builtin_huge_valf();

// per-warp shared-memory words; G = number of radii (runtime)
//   SLOT[64] | QROW[16] | MT 32x36 | queue 64x8 | THR[64][G] | HCNT[64][G] | HSUM[64][G]
#define G_SLOT(L) wsi[(L)]
#define G_MT(T, j) ws[80 + (T) * 36 + (j)]
#define G_QUEUE4(e) (reinterpret_cast<float4*>(ws + 80 + 32 * 36) + 2 * (e))
#define G_BASE (80 + 32 * 36 + kGQueue * 8)
#define G_THR(L, g) ws[G_BASE + (L) * G + (g)]
#define G_HCNT(L, g) wsi[G_BASE + 64 * G + (L) * G + (g)]
#define G_HSUM(L, g) ws[G_BASE + 128 * G + (L) * G + (g)]

__host__ __device__ inline int range_grid_warp_words(int G) { return G_BASE + 192 * G; }

__device__ __noinline__ void range_grid_refine(float* ws, int G, bool with_sum, int lane, int q, int N, int head,
                                               int n) {
    int* wsi = reinterpret_cast<int*>(ws);
    __syncwarp();
    float base = kGInf;
    float sq[kLow] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (lane < n) {
        const float4* e = G_QUEUE4((head + lane) % kGQueue);
        const float4 a = e[0], b = e[1];
        const int cand = __float_as_int(a.x);
        base = a.y; sq[0] = a.z; sq[1] = a.w;
        sq[2] = b.x; sq[3] = b.y; sq[4] = b.z; sq[5] = b.w;
        if (cand == q || cand >= N) base = kGInf;   // self by index (A4), padding rows (A19)
    }
    float X8[8];
    X8[0] = base;
#pragma unroll
    for (int u = 1; u < 8; ++u) {
        const int hb = 31 - __clz(u);
        X8[u] = __fadd_rn(X8[u & ~(1 << hb)], sq[2 + hb]);
    }
#pragma unroll
    for (int half = 0; half < 2; ++half) {
#pragma unroll
        for (int uu = 0; uu < 8; ++uu) {
            const float s0 = half ? __fadd_rn(X8[uu], sq[5]) : X8[uu];
            const float s1 = __fadd_rn(s0, sq[0]);
            const float s2 = __fadd_rn(s0, sq[1]);
            const float s3 = __fadd_rn(s1, sq[1]);
            G_MT(4 * uu + 0, lane) = s0;
            G_MT(4 * uu + 1, lane) = s1;
            G_MT(4 * uu + 2, lane) = s2;
            G_MT(4 * uu + 3, lane) = s3;
        }
        __syncwarp();
        const int T = 32 * half + lane;
        const float thr = G_THR(T, G - 1);   // the largest radius of this list (-1 for unused slots)
        unsigned mask = 0u;
#pragma unroll
        for (int j4 = 0; j4 < 8; ++j4) {
            const float4 m = *reinterpret_cast<const float4*>(&G_MT(lane, 4 * j4));
            mask |= (m.x < thr ? 1u : 0u) << (4 * j4);
            mask |= (m.y < thr ? 1u : 0u) << (4 * j4 + 1);
            mask |= (m.z < thr ? 1u : 0u) << (4 * j4 + 2);
            mask |= (m.w < thr ? 1u : 0u) << (4 * j4 + 3);
        }
#pragma unroll 1
        while (mask) {
            const int j = __ffs(mask) - 1;
            mask &= mask - 1u;
            const float d2 = G_MT(lane, j);
            int g = 0;   // smallest radius that contains the neighbour (radii ascend)
            while (!(d2 < G_THR(T, g))) ++g;
            G_HCNT(T, g) += 1;
            if (with_sum) G_HSUM(T, g) += sqrtf(d2);
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
    const long long n_items = static_cast<long long>(p.N) * p.n_batches;
    const unsigned lt = (1u << lane) - 1u;
    const int n_blocks = p.n_blocks;
    for (;;) {
        long long item = 0;
        if (lane == 0) item = atomicAdd(p.work_counter, 1ull);
        item = __shfl_sync(kFull, item, 0);
        if (item >= n_items) break;
        const int q = static_cast<int>(item % p.N);
        const int b = static_cast<int>(item / p.N);
        float qlo[kLow], qhi[9];
        {
            const float* qr = p.Xp + static_cast<size_t>(q) * kRowFloats;
#pragma unroll
            for (int j = 0; j < kLow; ++j) qlo[j] = qr[j];
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
        }
        __syncwarp();
        const bool g0_both = (G_SLOT(0) < 0) & (G_SLOT(1) < 0) & (G_SLOT(2) < 0);
        float Gm[16];
#pragma unroll
        for (int u = 0; u < 16; ++u)
            Gm[u] = fmaxf(fmaxf(G_THR(4 * u, G - 1), G_THR(4 * u + 1, G - 1)),
                          fmaxf(G_THR(4 * u + 2, G - 1), G_THR(4 * u + 3, G - 1)));
        float wq[9], w[9];
#pragma unroll
        for (int j = 0; j < 9; ++j) {
            w[j] = ((H >> (kLow + j)) & 1u) ? 1.f : 0.f;
            wq[j] = w[j] * qhi[j];
        }
        int qhead = 0, qtail = 0;
        float4 n0, n1, n2, n3;
        {
            const float4* b_ = p.Xb + lane;
            n0 = __ldg(b_); n1 = __ldg(b_ + 32); n2 = __ldg(b_ + 64); n3 = __ldg(b_ + 96);
        }
#pragma unroll 1
        for (int t = 0; t < n_blocks; ++t) {
            const float4 r0 = n0, r1 = n1, r2 = n2, r3 = n3;
            if (t + 1 < n_blocks) {
                const float4* b_ = p.Xb + static_cast<size_t>(t + 1) * 128 + lane;
                n0 = __ldg(b_); n1 = __ldg(b_ + 32); n2 = __ldg(b_ + 64); n3 = __ldg(b_ + 96);
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
            float X[16];
            X[0] = base;
#pragma unroll
            for (int u = 1; u < 16; ++u) {
                const int hb = 31 - __clz(u);
                X[u] = __fadd_rn(X[u & ~(1 << hb)], sq[2 + hb]);
            }
            float x0 = X[0];
            if (g0_both) x0 = __fadd_rn(__fadd_rn(X[0], sq[0]), sq[1]);
            bool pass = x0 < Gm[0];
#pragma unroll
            for (int u = 1; u < 16; ++u) pass |= (X[u] < Gm[u]);
            const unsigned bal = __ballot_sync(kFull, pass);
            if (bal) {
                if (pass) {
                    float4* e = G_QUEUE4((qtail + __popc(bal & lt)) % kGQueue);
                    e[0] = make_float4(__int_as_float(t * 32 + lane), base, sq[0], sq[1]);
                    e[1] = make_float4(sq[2], sq[3], sq[4], sq[5]);
                }
                qtail += __popc(bal);
                if (qtail - qhead >= 32) {
                    range_grid_refine(ws, G, with_sum, lane, q, p.N, qhead, 32);
                    qhead += 32;
                }
            }
        }
        if (qtail > qhead) range_grid_refine(ws, G, with_sum, lane, q, p.N, qhead, qtail - qhead);
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
                const size_t o = (static_cast<size_t>(sl) * G + g) * static_cast<size_t>(p.N) + q;
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
