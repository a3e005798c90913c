// grid_join.cu -- kNN self-join and eps range self-join of ONE feature subspace through the grid
// index of grid_index.cu: the engine for arbitrary mask lists, large N and large k.
//
// What it computes: PAPER.md:112, 122 (kNNSJ), PAPER.md:111, 154-156 (DSSJ), scores of
// the same outputs as the sub-lattice kernels.  How:
//   * one warp = 32 queries that are neighbours in cell order (lane = query); warps are independent
//     (no block-level synchronisation anywhere);
//   * the warp walks the (dim 0, dim 1) rows of the grid outwards from its home cell; for a row, each
//     lane forms the exact lower bound of every distance into that row (the distance chain with the
//     non-index terms dropped: rounding is monotone, so the bound holds for the computed fp32 values),
//     and from its current threshold the range of dim-2 bins a neighbour can still sit in; the union
//     of the lanes' ranges is one contiguous run of the cell-sorted compact table;
//   * the run streams through a per-warp shared-memory tile (coalesced 128-bit loads, next tile
//     prefetched into registers); every lane evaluates every candidate of the tile with broadcast
//     128-bit shared-memory reads: d FSUB + d FFMA + one compare per pair;
//   * kNN: per-lane max-heap of (d^2, id) in shared memory (conflict-free: entry e of lane l at
//     e*32 + l; for k > 256 in the lane's own rows of the output lists), root = threshold; a window of
//     the sorted order around the warp seeds the heaps first; heapsort at the end; ties by the smaller
//     id (reading A3);
//   * DSSJ: per-lane count and sum in registers (or G counters for a radius grid).
// The distance of a pair is the FMA chain over the mask's features in ascending order, the same
// wherever it is formed, so results do not depend on the grid resolution or the scan order
// (the DSSJ distance sums are accumulated in scan order, which is fixed by N and the mask).
#include "grid_join.cuh"

namespace snaps {

namespace {

constexpr int MODE_KNN = 0, MODE_RANGE = 1, MODE_RANGE_GRID = 2, MODE_KNN_BIG = 3;

// Warps per CTA.  The warps are independent and their running times differ widely (a warp of outliers
// walks many more rows), so a CTA holds its registers and shared memory until its slowest warp is done:
// with 8 warps per CTA 12.6 warps per SM were active on average where 16-24 fit.  Measured on config 5's
// masks at N = 10^6 (join kernels, 64 masks): kNN 9.04 s with 8 warps, 7.45 s with 2, 6.83 s with 1;
// DSSJ 2.46 / 1.92 / 1.99 s.
__host__ __device__ constexpr int warps_per_cta(int mode) { return (mode == MODE_KNN || mode == MODE_KNN_BIG) ? 1 : 2; }
constexpr int kTile = 64;            // candidates per tile
constexpr int kSeedHalf = 112;       // seed window: this many sorted positions either side of the warp
constexpr int kMaxG = 32;

__host__ __device__ constexpr int dp_of(int d) { return (d + 3) / 4 * 4; }

// per-warp shared-memory floats
__host__ __device__ constexpr int warp_words(int d, int mode, int k, int G) {
    return kTile * dp_of(d) + (mode == MODE_KNN ? 64 * k : 0) + (mode == MODE_RANGE_GRID ? 64 * G + 32 : 0);
}

// Per-lane max-heap of (d^2, id).  BIG = false: in shared memory, entry e of lane l at e*32 + l (conflict-free
// whatever path each lane's sift takes).  BIG = true (k > 256): in the lane's own rows of the output lists
// (out_dist / out_idx of its query), which the heapsort at the end leaves in their final ascending order.
template <bool BIG>
struct Heap {
    float* d;
    int* i;
    int lane;
    __device__ __forceinline__ float& D(int e) { return BIG ? d[e] : d[e * 32 + lane]; }
    __device__ __forceinline__ int& I(int e) { return BIG ? i[e] : i[e * 32 + lane]; }
    // replace the root (the largest key) by (v, id) and restore the heap over entries [0, n)
    __device__ __forceinline__ void sift(float v, int id, int n) {
        int e = 0;
        for (;;) {
            const int l = 2 * e + 1;
            if (l >= n) break;
            int c = l;
            float dc = D(l);
            int ic = I(l);
            if (l + 1 < n) {
                const float dr = D(l + 1);
                const int ir = I(l + 1);
                if (dr > dc || (dr == dc && ir > ic)) { c = l + 1; dc = dr; ic = ir; }
            }
            if (dc > v || (dc == v && ic > id)) {
                D(e) = dc;
                I(e) = ic;
                e = c;
            } else {
                break;
            }
        }
        D(e) = v;
        I(e) = id;
    }
};

// Packed fp32 pairs (sm_100: add.rn.f32x2 / fma.rn.f32x2 -> SASS FADD2 / FFMA2): two IEEE
// round-to-nearest results per instruction, bit-identical to the scalar operations.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

template <int D, int MODE>
__global__ void __launch_bounds__(warps_per_cta(MODE) * 32) grid_join_kernel(const GridJoinParams p) {
    constexpr int DP = dp_of(D);
    constexpr int G4 = DP / 2;                     // float4 per pair of candidates: two columns x two objects
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long slot = static_cast<long long>(blockIdx.x) * (blockDim.x >> 5) + warp;
    if (slot * 32 >= p.nq) return;                 // warps are independent: no block barrier exists
    const long long wid = p.warp_order ? p.warp_order[slot] : slot;
    const long long qi0 = wid * 32;
    const int k = p.k;
    float* wsm = reinterpret_cast<float*>(smem_raw) + static_cast<size_t>(warp) * warp_words(D, MODE, k, p.G);
    float4* tile4 = reinterpret_cast<float4*>(wsm);
    constexpr bool KNN = MODE == MODE_KNN || MODE == MODE_KNN_BIG;
    constexpr bool BIG = MODE == MODE_KNN_BIG;
    Heap<BIG> hp;
    hp.d = wsm + kTile * DP;
    hp.i = reinterpret_cast<int*>(hp.d + 32 * k);
    hp.lane = lane;
    // radius grid: per-lane histogram of hits by smallest radius, distance sums beside it
    int* gcnt = reinterpret_cast<int*>(wsm + kTile * DP);
    float* gsum = wsm + kTile * DP + 32 * p.G;
    float* gthr = wsm + kTile * DP + 64 * p.G;

    const GridPlan* pl = p.plan;
    const int N = p.N;
    const bool valid = qi0 + lane < p.nq;
    const int pos = valid ? (p.qlist ? p.qlist[qi0 + lane] : static_cast<int>(qi0) + lane) : -1;
    float q[D];
#pragma unroll
    for (int j = 0; j < D; ++j) q[j] = 0.f;
    uint32_t key = 0;
    int my_id = -1;
    if (valid) {
        key = p.keys[pos];
        my_id = p.perm[pos];
        if (BIG) {
            hp.d = p.out_dist + static_cast<size_t>(my_id - p.q_begin) * k;
            hp.i = p.out_idx + static_cast<size_t>(my_id - p.q_begin) * k;
        }
        const float* row = p.Xp + static_cast<size_t>(my_id) * kRowFloats;
#pragma unroll
        for (int j = 0; j < D; ++j) q[j] = __ldg(row + pl->feat[j]);
    }
    f32x2 nq[D];                                   // (-q_j, -q_j): c - q = c + (-q), the same rounding
#pragma unroll
    for (int j = 0; j < D; ++j) nq[j] = pack2(-q[j], -q[j]);
    // the lane's own bins and coordinates in the three grid dimensions
    const int b0 = p.bits[0], b1 = p.bits[1], b2 = p.bits[2];
    int my[3];
    my[2] = key & ((1u << b2) - 1u);
    my[1] = (key >> b2) & ((1u << b1) - 1u);
    my[0] = (key >> (b1 + b2)) & ((1u << b0) - 1u);
    const float* E[3];
    float qx[3];
#pragma unroll
    for (int g = 0; g < 3; ++g) {
        const int f = pl->idx_feat[g];
        E[g] = p.edges + static_cast<size_t>(f < 0 ? 0 : f) * kGridEdgeStride;
        const int col = pl->idx_col[g];
        float v = 0.f;
#pragma unroll
        for (int j = 0; j < D; ++j) v = (j == col) ? q[j] : v;
        qx[g] = v;
    }
    // home cell = the middle lane's (lane 0's if the warp is not full); spans of the lanes' bins
    const int src = (qi0 + 16 < p.nq) ? 16 : 0;
    int home[3], mn[3], mx[3];
#pragma unroll
    for (int g = 0; g < 3; ++g) {
        home[g] = __shfl_sync(kFull, my[g], src);
        const int v = valid ? my[g] : home[g];
        mn[g] = __reduce_min_sync(kFull, v);
        mx[g] = __reduce_max_sync(kFull, v);
    }

    // ---- per-lane state
    float tau = valid ? __int_as_float(0x7f800000) : -1.f;   // pass test: d^2 <= tau
    int tau_id = 0x7fffffff;
    int cnt = 0;
    float sum = 0.f;
    if (KNN) {
        if (!BIG || valid)
            for (int e = 0; e < k; ++e) {
                hp.D(e) = __int_as_float(0x7f800000);
                hp.I(e) = 0x7fffffff;
            }
    } else if (MODE == MODE_RANGE) {
        if (valid) tau = p.eps2;
    } else {
        for (int g = 0; g < p.G; ++g) {
            gcnt[g * 32 + lane] = 0;
            gsum[g * 32 + lane] = 0.f;
        }
        if (lane < p.G) gthr[lane] = p.eps2_grid[lane];
        if (valid) tau = p.eps2_grid[p.G - 1];
    }
    __syncwarp();

    float g_first = 0.f, g_per_eps = 0.f;                    // radius grid: first radius and bins per unit of distance
    if (MODE == MODE_RANGE_GRID) {
        g_first = sqrtf(fmaxf(gthr[0], 0.f));
        const float g_last = sqrtf(fmaxf(gthr[p.G - 1], 0.f));
        g_per_eps = (p.G > 1 && g_last > g_first) ? static_cast<float>(p.G - 1) / (g_last - g_first) : 0.f;
    }

    // ---- one candidate against this lane's query
    auto consider = [&](float acc, int cpos) {
        if (KNN) {
            if (cpos == pos) return;                         // self by index (reading A4)
            const int id = __ldg(p.perm + cpos);
            if (acc < tau || id < tau_id) {
                hp.sift(acc, id, k);
                tau = hp.D(0);
                tau_id = hp.I(0);
            }
        } else if (MODE == MODE_RANGE) {
            if (cpos == pos) return;
            cnt += 1;
            sum += sqrtf(acc);
        } else {
            if (cpos == pos) return;
            // smallest radius that contains the pair: guessed as if the radii were evenly spaced (the library's own
            // grids are, reading A22), settled against the exact thresholds on either side -- any grid stays exact
            const float dd = sqrtf(acc);
            int g = min(max(__float2int_ru((dd - g_first) * g_per_eps), 0), p.G - 1);
            if (g > 0 && acc <= gthr[g - 1]) {
                --g;
                while (g > 0 && acc <= gthr[g - 1]) --g;
            } else {
                while (acc > gthr[g]) ++g;                   // ends: acc <= the largest threshold
            }
            gcnt[g * 32 + lane] += 1;
            gsum[g * 32 + lane] += dd;
        }
    };

    // ---- stream sorted positions [a, b) through the tile; lanes with `active` evaluate them
    auto scan = [&](int a, int b, bool active) {
        if (a >= b) return;
        const bool any_active = __any_sync(kFull, active);
        if (!any_active) return;
        // pairs of sorted positions (2i, 2i+1): [pa, pb) covers [a, b); the stray position at either end
        // is evaluated and dropped by the range test below
        const int pa = a >> 1, pb = (b + 1) >> 1;
        constexpr int kTilePairs = kTile / 2;
        constexpr int PF = (kTilePairs * G4 + 31) / 32;      // float4 per lane per tile
        float4 nx[PF];
        auto fetch = [&](int t0) {
            const int n4 = min(kTilePairs, pb - t0) * G4;
            const float4* srcp = reinterpret_cast<const float4*>(p.Xs) + static_cast<size_t>(t0) * G4;
#pragma unroll
            for (int u = 0; u < PF; ++u) {
                const int i = lane + 32 * u;
                if (i < n4) nx[u] = __ldg(srcp + i);
            }
        };
        fetch(pa);
        for (int t0 = pa; t0 < pb; t0 += kTilePairs) {
            const int n = min(kTilePairs, pb - t0);
            __syncwarp();
#pragma unroll
            for (int u = 0; u < PF; ++u) {
                const int i = lane + 32 * u;
                if (i < n * G4) tile4[i] = nx[u];
            }
            __syncwarp();
            if (t0 + kTilePairs < pb) fetch(t0 + kTilePairs);
            if (active) {
#pragma unroll 2
                for (int r = 0; r < n; ++r) {
                    f32x2 acc = 0ull;                        // (0.f, 0.f)
#pragma unroll
                    for (int g = 0; g < G4; ++g) {
                        const float4 v = tile4[r * G4 + g];  // columns 2g, 2g+1 of candidates 2(t0+r), 2(t0+r)+1
                        if (2 * g < D) {
                            const f32x2 diff = add2(pack2(v.x, v.y), nq[2 * g]);
                            acc = fma2(diff, diff, acc);
                        }
                        if (2 * g + 1 < D) {
                            const f32x2 diff = add2(pack2(v.z, v.w), nq[2 * g + 1 < D ? 2 * g + 1 : 0]);
                            acc = fma2(diff, diff, acc);
                        }
                    }
                    float a0, a1;
                    unpack2(acc, a0, a1);
                    if (a0 <= tau || a1 <= tau) {
                        const int c0 = 2 * (t0 + r);
                        if (a0 <= tau && c0 >= a) consider(a0, c0);
                        if (a1 <= tau && c0 + 1 < b) consider(a1, c0 + 1);
                    }
                }
            }
        }
        __syncwarp();
    };

    // ---- kNN: seed the heaps from the sorted neighbourhood of the warp
    int w0 = 0, w1 = 0;
    if (KNN) {
        const int p_first = __shfl_sync(kFull, pos, 0);
        const int n_valid = min(32, static_cast<int>(p.nq - qi0));
        const int p_last = __shfl_sync(kFull, pos, n_valid - 1);
        const int half_w = max(kSeedHalf, k);        // enough positions to fill every heap
        w0 = max(0, p_first - half_w);
        w1 = min(N, p_last + 1 + half_w);
        scan(w0, w1, valid);
    }

    // lower bound of |x - q| over bin s of dimension g for this lane (0 inside the lane's own bin)
    auto slab_gap = [&](int g, int bits, int s) -> float {
        if (bits == 0 || s == my[g]) return 0.f;
        const int sh = kGridMasterBits - bits;
        return s > my[g] ? __fsub_rn(__ldg(E[g] + (s << sh)), qx[g]) : __fsub_rn(qx[g], __ldg(E[g] + ((s + 1) << sh)));
    };
    // bin of dimension 2 (at its resolution) that holds value v
    auto bin2_of = [&](float v) -> int {
        const int sh = kGridMasterBits - b2;
        int lo = 0, hi = 1 << b2;
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(E[2] + (mid << sh)) <= v) lo = mid + 1; else hi = mid;
        }
        return lo > 0 ? lo - 1 : 0;
    };

    // ---- rows outwards from the home cell
    const int B0 = 1 << b0, B1 = 1 << b1;
    bool up0 = true, dn0 = true;
    for (int o0 = 0; o0 < B0 && (up0 || dn0); ++o0) {
#pragma unroll 1
        for (int side0 = 0; side0 < 2; ++side0) {
            if (side0 == 1 && o0 == 0) continue;
            bool& live0 = side0 == 0 ? up0 : dn0;
            if (!live0) continue;
            const int s0 = side0 == 0 ? home[0] + o0 : home[0] - o0;
            if (s0 < 0 || s0 >= B0) { live0 = false; continue; }
            const float g0 = slab_gap(0, b0, s0);
            const float lb0 = __fmul_rn(g0, g0);
            const bool alive0 = valid && lb0 <= tau;
            if (!__any_sync(kFull, alive0)) {
                if (side0 == 0 ? s0 > mx[0] : s0 < mn[0]) live0 = false;   // bounds only grow from here on
                continue;
            }
            bool up1 = true, dn1 = true;
            for (int o1 = 0; o1 < B1 && (up1 || dn1); ++o1) {
#pragma unroll 1
                for (int side1 = 0; side1 < 2; ++side1) {
                    if (side1 == 1 && o1 == 0) continue;
                    bool& live1 = side1 == 0 ? up1 : dn1;
                    if (!live1) continue;
                    const int s1 = side1 == 0 ? home[1] + o1 : home[1] - o1;
                    if (s1 < 0 || s1 >= B1) { live1 = false; continue; }
                    const float g1 = slab_gap(1, b1, s1);
                    const float lb01 = __fmaf_rn(g1, g1, lb0);
                    const bool alive = valid && lb01 <= tau;
                    int lo = 0x7fffffff, hi = -1;
                    if (alive) {
                        // a candidate of this row can pass only if fl(diff2^2 + lb01) <= tau; with four
                        // ulps of slack that needs |x2 - q2| <= rho (see DESIGN.md for the rounding argument)
                        const float budget = fmaxf(__fsub_ru(__fmul_ru(tau, 1.00000024f), lb01), 0.f);
                        const float rho = __fmul_ru(__fsqrt_ru(budget), 1.0000005f);
                        lo = b2 ? bin2_of(__fsub_rd(qx[2], rho)) : 0;
                        hi = b2 ? bin2_of(__fadd_ru(qx[2], rho)) : 0;
                    }
                    if (!__any_sync(kFull, alive)) {
                        if (side1 == 0 ? s1 > mx[1] : s1 < mn[1]) live1 = false;
                        continue;
                    }
                    // The lanes' bin ranges are merged into clusters of overlapping or adjoining ranges and each
                    // cluster is scanned by its own lanes only: the lanes of a warp that straddles the end of one
                    // grid row and the start of the next sit at opposite ends of dimension 2, and the hull of
                    // their ranges would be the whole row.
                    const int cell = ((s0 << b1) | s1) << b2;
                    bool todo = alive;
                    while (true) {
                        const unsigned rem = __ballot_sync(kFull, todo);
                        if (!rem) break;
                        const int lead = __ffs(rem) - 1;
                        int L = __shfl_sync(kFull, lo, lead), H = __shfl_sync(kFull, hi, lead);
                        bool in = false;
                        while (true) {
                            in = todo && lo <= H + 1 && hi >= L - 1;
                            const int nL = __reduce_min_sync(kFull, in ? lo : L);
                            const int nH = __reduce_max_sync(kFull, in ? hi : H);
                            if (nL == L && nH == H) break;
                            L = nL;
                            H = nH;
                        }
                        const int a = __ldg(p.cell_start + cell + L);
                        const int b = __ldg(p.cell_start + cell + H + 1);
                        // the seed window has been evaluated already
                        scan(a, min(b, w0), in);
                        scan(max(a, w1), b, in);
                        todo = todo && !in;
                    }
                }
            }
        }
    }

    // ---- a7: emit
    if (!valid) return;
    if (KNN) {
        // heapsort: ascending by (d^2, id) in entries 0..k-1
        for (int n = k - 1; n >= 1; --n) {
            const float v = hp.D(n);
            const int id = hp.I(n);
            hp.D(n) = hp.D(0);
            hp.I(n) = hp.I(0);
            hp.sift(v, id, n);
        }
        const size_t o = static_cast<size_t>(my_id - p.q_begin);
        float s = 0.f, dk = 0.f;
        for (int e = 0; e < k; ++e) {
            const float dd = sqrtf(hp.D(e));
            const int id = hp.I(e);
            s += dd;
            dk = dd;
            if (BIG) {
                hp.D(e) = dd;                                 // the heap rows ARE the output lists
            } else {
                if (p.out_idx) p.out_idx[o * k + e] = id;
                if (p.out_dist) p.out_dist[o * k + e] = dd;
            }
            if (p.out_indeg) atomicAdd(&p.out_indeg[id], 1);
        }
        if (p.out_kth) p.out_kth[o] = dk;
        if (p.out_mean) p.out_mean[o] = s / static_cast<float>(k);
    } else if (MODE == MODE_RANGE) {
        const size_t o = static_cast<size_t>(my_id - p.q_begin);
        p.out_count[o] = static_cast<uint32_t>(cnt);
        if (p.out_sum) p.out_sum[o] = sum;
        if (p.out_rmean) p.out_rmean[o] = cnt > 0 ? sum / static_cast<float>(cnt) : 0.f;   // reading A6
    } else {
        // cumulative over the ascending radii (A(eps_j) is nested in A(eps_j+1))
        int c = 0;
        float s = 0.f;
        for (int g = 0; g < p.G; ++g) {
            c += gcnt[g * 32 + lane];
            s += gsum[g * 32 + lane];
            const size_t o = static_cast<size_t>(g) * p.nq + static_cast<size_t>(my_id - p.q_begin);
            p.out_count[o] = static_cast<uint32_t>(c);
            if (p.out_sum) p.out_sum[o] = s;
            if (p.out_rmean) p.out_rmean[o] = c > 0 ? s / static_cast<float>(c) : 0.f;
        }
    }
}

template <int MODE, int D>
cudaError_t launch_d(const GridJoinParams& p, cudaStream_t st) {
    const size_t per_warp = static_cast<size_t>(warp_words(D, MODE, p.k, p.G)) * 4;
    int wpc = warps_per_cta(MODE);
    while (wpc > 1 && wpc * per_warp > 200 * 1024) --wpc;
    const size_t smem = wpc * per_warp;
    auto kernel = grid_join_kernel<D, MODE>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
        if (e != cudaSuccess) return e;
    }
    const long long warps = (static_cast<long long>(p.nq) + 31) / 32;
    const int grid = static_cast<int>((warps + wpc - 1) / wpc);
    kernel<<<grid, wpc * 32, smem, st>>>(p);
    return cudaGetLastError();
}

template <int MODE>
cudaError_t launch_mode(const GridJoinParams& p, int d, cudaStream_t st) {
    switch (d) {
        case 1: return launch_d<MODE, 1>(p, st);
        case 2: return launch_d<MODE, 2>(p, st);
        case 3: return launch_d<MODE, 3>(p, st);
        case 4: return launch_d<MODE, 4>(p, st);
        case 5: return launch_d<MODE, 5>(p, st);
        case 6: return launch_d<MODE, 6>(p, st);
        case 7: return launch_d<MODE, 7>(p, st);
        case 8: return launch_d<MODE, 8>(p, st);
        case 9: return launch_d<MODE, 9>(p, st);
        case 10: return launch_d<MODE, 10>(p, st);
        case 11: return launch_d<MODE, 11>(p, st);
        case 12: return launch_d<MODE, 12>(p, st);
        case 13: return launch_d<MODE, 13>(p, st);
        case 14: return launch_d<MODE, 14>(p, st);
        case 15: return launch_d<MODE, 15>(p, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t grid_knn_launch(const GridJoinParams& p, int d, cudaStream_t st) {
    if (p.k < 1 || p.k > kGridMaxKBig) return cudaErrorInvalidValue;
    if (p.k > kGridMaxK) {
        if (!p.out_idx || !p.out_dist) return cudaErrorInvalidValue;   // the heaps live in the output lists
        return launch_mode<MODE_KNN_BIG>(p, d, st);
    }
    return launch_mode<MODE_KNN>(p, d, st);
}

cudaError_t grid_range_launch(const GridJoinParams& p, int d, cudaStream_t st) {
    if (p.G > 0) {
        if (p.G > kMaxG) return cudaErrorInvalidValue;
        return launch_mode<MODE_RANGE_GRID>(p, d, st);
    }
    return launch_mode<MODE_RANGE>(p, d, st);
}

}  // namespace snaps
