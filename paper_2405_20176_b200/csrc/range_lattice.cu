// range_lattice.cu -- eps range self-join (DSSJ) over a batch of feature subspaces
// (steps a3, a4, a6, a7).
//
// What it computes: PAPER.md:111, 154-156: for every object i and mask S the number of
// objects j != i with D(i,j;S) <= eps_S and the sum of those D
// (PAPER.md:165).  Same pair staging and add-only subset sums as knn_lattice.cu; the
// thresholds are the per-mask constants eps_S^2 (held in registers, one per lattice slot),
// so no list state exists: a warp vote per group of 4 sums gates the counting path, where
// a ballot's popcount is added to the list's counter by lane 0 (the warp-aggregated form
// of an atomic increment) and each lane adds sqrt(d^2) to its own partial sum, reduced in
// lane order at the end of the batch (deterministic).
#include "range_lattice.cuh"

namespace snaps {

#define R_CNT(L) wsi[(L)]
#define R_SLOT(L) wsi[64 + (L)]
#define R_SUM(L, ln) ws[128 + (L) * 33 + (ln)]

#define COUNT_ONE(sval, Lidx)                                                 \
    {                                                                         \
        const bool in_ = (sval) < thr[Lidx];                                  \
        const unsigned bal_ = __ballot_sync(kFull, in_);                      \
        if (bal_) {                                                           \
            if (lane == 0) R_CNT(Lidx) += __popc(bal_);                       \
            if (WITH_SUM && in_) R_SUM(Lidx, lane) += sqrtf(sval);            \
        }                                                                     \
    }

template <bool WITH_SUM>
__global__ void __launch_bounds__(kRangeMaxThreads, 1) range_lattice_kernel(const RangeParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    float* tiles = reinterpret_cast<float*>(smem);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + kStages * kTileBytes);
    uint64_t* empty = full + kStages;
    int* s_item = reinterpret_cast<int*>(empty + kStages);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int W = p.warps;
    const int ws_floats = 128 + (WITH_SUM ? 64 * 33 : 0);
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

    uint32_t g = 0;
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
        }
#pragma unroll 1
        for (int b = b0; b < b1; ++b) {
            const BatchDesc* bd = &p.batches[b];
            const uint32_t H = bd->hmask;
            float thr[kLat];
            {
                const float4* t4 = reinterpret_cast<const float4*>(bd->thr);
#pragma unroll
                for (int i4 = 0; i4 < 16; ++i4) {
                    const float4 v = t4[i4];
                    thr[4 * i4 + 0] = v.x;
                    thr[4 * i4 + 1] = v.y;
                    thr[4 * i4 + 2] = v.z;
                    thr[4 * i4 + 3] = v.w;
                }
            }
            __syncwarp();
            for (int h = 0; h < 2; ++h) {
                const int L = lane + 32 * h;
                R_CNT(L) = 0;
                R_SLOT(L) = bd->slot[L];
            }
            if (WITH_SUM)
                for (int L = 0; L < kLat; ++L) R_SUM(L, lane) = 0.f;
            __syncwarp();
            float wq[9], w[9];
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
                        if (cand >= p.N || cand == q) base = __int_as_float(0x7f800000);
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
                                COUNT_ONE(s0, 4 * u + 0)
                                COUNT_ONE(s1, 4 * u + 1)
                                COUNT_ONE(s2, 4 * u + 2)
                                COUNT_ONE(s3, 4 * u + 3)
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[s]);
            }
            if (active) {
                __syncwarp();
                for (int h = 0; h < 2; ++h) {
                    const int L = lane + 32 * h;
                    const int sl = R_SLOT(L);
                    if (sl < 0) continue;
                    const size_t o = static_cast<size_t>(sl) * static_cast<size_t>(p.N) + q;
                    const int cnt = R_CNT(L);
                    p.out_count[o] = static_cast<uint32_t>(cnt);
                    if (WITH_SUM) {
                        float tot = 0.f;
                        for (int ln = 0; ln < 32; ++ln) tot += R_SUM(L, ln);
                        if (p.out_sum) p.out_sum[o] = tot;
                        if (p.out_mean) p.out_mean[o] = cnt > 0 ? tot / static_cast<float>(cnt) : 0.f;
                    }
                }
                __syncwarp();
            }
        }
    }
}

size_t range_lattice_smem_bytes(int warps, bool with_sum) {
    return static_cast<size_t>(kStages) * kTileBytes + 128 +
           static_cast<size_t>(warps) * (128 + (with_sum ? 64 * 33 : 0)) * 4;
}

cudaError_t range_lattice_launch(const RangeParams& p, int grid, cudaStream_t stream) {
    const bool with_sum = p.out_sum != nullptr || p.out_mean != nullptr;
    const size_t smem = range_lattice_smem_bytes(p.warps, with_sum);
    cudaError_t e;
    if (with_sum) {
        e = cudaFuncSetAttribute(range_lattice_kernel<true>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        range_lattice_kernel<true><<<grid, (p.warps + 1) * 32, smem, stream>>>(p);
    } else {
        e = cudaFuncSetAttribute(range_lattice_kernel<false>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        range_lattice_kernel<false><<<grid, (p.warps + 1) * 32, smem, stream>>>(p);
    }
    return cudaGetLastError();
}

}  // namespace snaps
