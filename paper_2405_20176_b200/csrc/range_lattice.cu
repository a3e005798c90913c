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
//   * COMPACT passing candidates into a per-warp queue; REFINE every 32 of them: lane = candidate
//     forms the 64 subset sums (add-only, fixed order), a 32 x 32 shared-memory transpose hands
//     them to the list owners (lane = list), which count the sums below eps^2 with one popcount
//     and add sqrt(d^2) of the hits to the list's running sum in candidate order (deterministic;
//     each list is touched by one lane only -- no atomics are needed at all).
#include "range_lattice.cuh"

namespace snaps {

constexpr int kRQueue = 64;  // queue entries of 8 words; refine as soon as 32 are waiting
constexpr float kRInf = __builtin_huge_valf();

// per-warp shared-memory words
#define R_THR(L) ws[(L)]
#define R_SLOT(L) wsi[64 + (L)]
#define R_CNT(L) wsi[128 + (L)]
#define R_SUM(L) ws[192 + (L)]
#define R_QROW(j) ws[256 + (j)]
#define R_MT(T, j) ws[272 + (T) * 36 + (j)]
#define R_QUEUE4(e) (reinterpret_cast<float4*>(ws + 272 + 32 * 36) + 2 * (e))

__host__ __device__ constexpr int range_warp_words() { return 272 + 32 * 36 + kRQueue * 8; }

template <bool WITH_SUM>
__device__ __noinline__ void range_refine(float* ws, int lane, int q, int N, int head, int n) {
    int* wsi = reinterpret_cast<int*>(ws);
    __syncwarp();
    float base = kRInf;
    float sq[kLow] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (lane < n) {
        const float4* e = R_QUEUE4((head + lane) % kRQueue);
        const float4 a = e[0], b = e[1];
        const int cand = __float_as_int(a.x);
        base = a.y; sq[0] = a.z; sq[1] = a.w;
        sq[2] = b.x; sq[3] = b.y; sq[4] = b.z; sq[5] = b.w;
        // self by index (reading A4) and padding rows (A19) are never counted
        if (cand == q || cand >= N) base = kRInf;
    }
    float X8[8];   // partial sums over features 2,3,4; feature 5 is added per half
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
            R_MT(4 * uu + 0, lane) = s0;
            R_MT(4 * uu + 1, lane) = s1;
            R_MT(4 * uu + 2, lane) = s2;
            R_MT(4 * uu + 3, lane) = s3;
        }
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

// SWEEP: the pivot sweep of pivot_sort.cu (large N): scan the copy sorted by the batch's lowest
// high feature outwards from the query, stop a direction once that feature alone is beyond the
// batch's largest eps^2 (thresholds are constants here, so the bound never moves).
template <bool WITH_SUM, bool SWEEP>
__global__ void __launch_bounds__(kRangeMaxThreads, 1) range_lattice_kernel(const RangeParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float* ws = reinterpret_cast<float*>(smem) + static_cast<size_t>(warp) * range_warp_words();
    int* wsi = reinterpret_cast<int*>(ws);
    const long long n_items = static_cast<long long>(p.N) * p.n_bchunks;
    const unsigned lt = (1u << lane) - 1u;
    const int n_blocks = p.n_blocks;
    for (;;) {
        long long item = 0;
        if (lane == 0) item = atomicAdd(p.work_counter, 1ull);
        item = __shfl_sync(kFull, item, 0);
        if (item >= n_items) break;
        const int q = static_cast<int>(item % p.N);
        const int bc = static_cast<int>(item / p.N);
        const int b0 = bc * p.batches_per_item;
        const int b1 = min(b0 + p.batches_per_item, p.n_batches);
        float qlo[kLow];
        float qhi[9];
        {
            const float* qr = p.Xp + static_cast<size_t>(q) * kRowFloats;
#pragma unroll
            for (int j = 0; j < kLow; ++j) qlo[j] = qr[j];
#pragma unroll
            for (int j = 0; j < 9; ++j) qhi[j] = qr[kLow + j];
            __syncwarp();
            if (lane < 15) R_QROW(lane) = qr[lane];
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
            // group 0 = lattice slots {}, {0}, {1}, {0,1}: when only {0,1} is asked for, its own sum is
            // the group's bound (X[0] alone is 0 when H is empty and would let every candidate through)
            const bool g0_both = (R_SLOT(0) < 0) & (R_SLOT(1) < 0) & (R_SLOT(2) < 0);
            float G[16];   // group maxima of the (constant) thresholds
#pragma unroll
            for (int u = 0; u < 16; ++u) {
                const float4 t = *reinterpret_cast<const float4*>(&R_THR(4 * u));
                G[u] = fmaxf(fmaxf(t.x, t.y), fmaxf(t.z, t.w));
            }
            float wq[9], w[9];  // high features: diff = c*w - q*w, w in {0,1}
#pragma unroll
            for (int j = 0; j < 9; ++j) {
                w[j] = ((H >> (kLow + j)) & 1u) ? 1.f : 0.f;
                wq[j] = w[j] * qhi[j];
            }
            int qhead = 0, qtail = 0;
#define LOAD_BLOCK(dst, tab_, t_)                                                             \
    {                                                                                         \
        const float4* b_ = (tab_) + static_cast<size_t>(t_) * 128 + lane;                      \
        dst.v0 = __ldg(b_); dst.v1 = __ldg(b_ + 32); dst.v2 = __ldg(b_ + 64); dst.v3 = __ldg(b_ + 96); \
    }
#define FILTER_BLOCK(r, t_, CAND_)                                                            \
    {                                                                                         \
        const float c[15] = {r.v0.x, r.v0.y, r.v0.z, r.v0.w, r.v1.x, r.v1.y, r.v1.z, r.v1.w,   \
                             r.v2.x, r.v2.y, r.v2.z, r.v2.w, r.v3.x, r.v3.y, r.v3.z};          \
        float sq[kLow];                                                                       \
        _Pragma("unroll") for (int j = 0; j < kLow; ++j) {                                    \
            const float diff = c[j] - qlo[j];                                                 \
            sq[j] = __fmul_rn(diff, diff);                                                    \
        }                                                                                     \
        float base = 0.f;                                                                     \
        _Pragma("unroll") for (int j = 0; j < 9; ++j) {                                       \
            const float diff = __fmaf_rn(c[kLow + j], w[j], -wq[j]);                          \
            base = __fmaf_rn(diff, diff, base);                                               \
        }                                                                                     \
        float X[16];                                                                          \
        X[0] = base;                                                                          \
        _Pragma("unroll") for (int u = 1; u < 16; ++u) {                                      \
            const int hb = 31 - __clz(u);                                                     \
            X[u] = __fadd_rn(X[u & ~(1 << hb)], sq[2 + hb]);                                  \
        }                                                                                     \
        float x0 = X[0];                                                                      \
        if (g0_both) x0 = __fadd_rn(__fadd_rn(X[0], sq[0]), sq[1]);                           \
        bool pa = x0 < G[0], pb = false;                                                      \
        _Pragma("unroll") for (int u = 0; u < 16; u += 2) {                                   \
            if (u > 0) pa |= (X[u] < G[u]);                                                   \
            pb |= (X[u + 1] < G[u + 1]);                                                      \
        }                                                                                     \
        const bool pass = pa | pb;                                                            \
        const unsigned bal = __ballot_sync(kFull, pass);                                      \
        if (bal) {                                                                            \
            if (pass) {                                                                       \
                float4* e = R_QUEUE4((qtail + __popc(bal & lt)) % kRQueue);                   \
                e[0] = make_float4(__int_as_float(CAND_), base, sq[0], sq[1]);                \
                e[1] = make_float4(sq[2], sq[3], sq[4], sq[5]);                               \
            }                                                                                 \
            qtail += __popc(bal);                                                             \
            if (qtail - qhead >= 32) {                                                        \
                range_refine<WITH_SUM>(ws, lane, q, p.N, qhead, 32);                          \
                qhead += 32;                                                                  \
            }                                                                                 \
        }                                                                                     \
    }
            struct Blk { float4 v0, v1, v2, v3; };
            if (!SWEEP) {
                Blk ra, rb;
                LOAD_BLOCK(ra, p.Xb, 0)
                rb = ra;
#pragma unroll 1
                for (int t = 0; t < n_blocks; t += 2) {
                    if (t + 1 < n_blocks) LOAD_BLOCK(rb, p.Xb, t + 1)
                    FILTER_BLOCK(ra, t, (t) * 32 + lane)
                    if (t + 1 < n_blocks) {
                        if (t + 2 < n_blocks) LOAD_BLOCK(ra, p.Xb, t + 2)
                        FILTER_BLOCK(rb, t + 1, (t + 1) * 32 + lane)
                    }
                }
            } else {
                const int pf = bd->pivot;   // a feature all valid masks of the batch contain, or -1
                const float4* tab = pf >= 0 ? p.Xs[pf] : p.Xb;
                const int* idm = pf >= 0 ? p.idmap[pf] : nullptr;
                const float* pv = pf >= 0 ? p.piv[pf] : nullptr;
                const int t0 = pf >= 0 ? (p.pos[pf][q] >> 5) : 0;
                const float qf = pf >= 0 ? R_QROW(pf) : 0.f;
                float Gall = G[0];
#pragma unroll
                for (int u = 1; u < 16; ++u) Gall = fmaxf(Gall, G[u]);
#pragma unroll 1
                for (int dir = 1; dir >= -1; dir -= 2) {
                    int t = dir > 0 ? t0 : t0 - 1;
                    const int t_end = dir > 0 ? n_blocks : -1;
                    if (t != t_end) {
                        const int eo = dir > 0 ? 31 : 0;
                        Blk nx;
                        float pe_n = 0.f;
                        LOAD_BLOCK(nx, tab, t)
                        if (pv) pe_n = __ldg(pv + 32 * t + eo);
#pragma unroll 1
                        for (;;) {
                            const Blk r = nx;
                            const float pe = pe_n;
                            const int tn = t + dir;
                            if (tn != t_end) {
                                LOAD_BLOCK(nx, tab, tn)
                                if (pv) pe_n = __ldg(pv + 32 * tn + eo);
                            }
                            FILTER_BLOCK(r, t, (idm ? __ldg(idm + t * 32 + lane) : t * 32 + lane))
                            if (pv) {
                                const float de = dir > 0 ? pe - qf : qf - pe;
                                if (de > 0.f && __fmul_rn(de, de) >= Gall) break;
                            }
                            if (tn == t_end) break;
                            t = tn;
                        }
                    }
                    if (!pv) break;
                }
            }
#undef LOAD_BLOCK
#undef FILTER_BLOCK
            if (qtail > qhead) range_refine<WITH_SUM>(ws, lane, q, p.N, qhead, qtail - qhead);
            // ---- a7: counts, sums, means (0 when there is no neighbour: PAPER.md:266, reading A6)
            __syncwarp();
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int L = lane + 32 * h;
                const int sl = R_SLOT(L);
                if (sl < 0) continue;
                const size_t o = static_cast<size_t>(sl) * static_cast<size_t>(p.N) + q;
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
    auto kernel = p.sweep ? (with_sum ? range_lattice_kernel<true, true> : range_lattice_kernel<false, true>)
                          : (with_sum ? range_lattice_kernel<true, false> : range_lattice_kernel<false, false>);
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kernel<<<grid, p.warps * 32, smem, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace snaps
