// knn_bigk.cu -- kNN self-join of ONE feature subspace for long lists on small tables
// (384 < k <= 4096, N <= 131,072): PAPER.md:258, k_max = 4096 on SNAPShot1's 31,693 objects.
//
// At k = 13 % of N no index prunes anything, and a per-query heap of 4096 entries in global memory spends its
// time in divergent sifts (grid_join.cu's in-place mode: 400-490 ms per subspace at k = 4096; here 21-31 ms):
//   * SELECT: one CTA = 32 queries (lane = query; its four warps take alternate tiles) streams ALL candidates, the
//     distance of a pair formed by the same instruction sequence as in grid_join.cu (so both paths give the
//     same lists), and finds the query's k-th smallest key (d^2 bits << 17 | id) by radix selection: up to six passes
//     over the candidates, each a 256-bin per-lane histogram of the next 8 key bits among the candidates that
//     match the prefix so far.  Keys are unique (ids are), so the k-th key is exact and ties go to the smaller id
//     (reading A3); the passes stop once every lane's k-th key is the last of its bin (typically after three or
//     four).  A last pass writes the k keys <= the k-th, unordered;
//   * SORT: one CUB segmented radix sort of the nq segments of k keys (48 significant bits);
//   * FINALISE (a7): ids, sqrt, k-th and mean distance (summed in list order, as everywhere), in-degree.
// Every pass recomputes the distances: 7 N^2 d flops per subspace is milliseconds at this N, far less than
// keeping N distances per query anywhere.
#include "knn_bigk.cuh"

#include <cub/device/device_segmented_radix_sort.cuh>

namespace snaps {

namespace {

constexpr int kWarpsB = 4;            // warps per CTA = per group of 32 queries (they share the candidates out)
constexpr int kTileB = 64;            // candidates per tile
constexpr int kBins = 256;
constexpr int kIdBits = 17;

__host__ __device__ constexpr int dpb(int d) { return (d + 3) / 4 * 4; }
// per-warp shared-memory words; the per-lane histogram counts in 16 bits when no bin can overflow them (N < 65,536):
// half the footprint, twice the warps per SM
__host__ __device__ constexpr int warp_words_b(int d, int counter_bytes) { return kTileB * dpb(d) + kTileB + kBins * 8 * counter_bytes; }

typedef unsigned long long u64;

template <int D, typename C>
__global__ void __launch_bounds__(kWarpsB * 32) bigk_select_kernel(const GridJoinParams p, u64* __restrict__ keys_out) {
    constexpr int DP = dpb(D);
    constexpr int G4 = DP / 2;                     // float4 per pair of candidates
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // one CTA = one group of 32 queries; its kWarpsB warps take alternate candidate tiles and add up their
    // histograms (31,693 queries are only 991 groups: one warp each would leave the SMs half empty)
    const long long qi0 = static_cast<long long>(blockIdx.x) * 32;
    float* wsm = reinterpret_cast<float*>(smem_raw) + static_cast<size_t>(warp) * warp_words_b(D, sizeof(C));
    int* emit_cnt = reinterpret_cast<int*>(reinterpret_cast<float*>(smem_raw) + static_cast<size_t>(kWarpsB) * warp_words_b(D, sizeof(C)));
    float4* tile4 = reinterpret_cast<float4*>(wsm);
    int* tile_id = reinterpret_cast<int*>(wsm + kTileB * DP);
    C* hist = reinterpret_cast<C*>(wsm + kTileB * DP + kTileB);
    const GridPlan* pl = p.plan;
    const int N = p.N, k = p.k;
    const bool valid = qi0 + lane < p.nq;
    const int pos = valid ? (p.qlist ? p.qlist[qi0 + lane] : static_cast<int>(qi0) + lane) : -1;
    const int my_id = valid ? p.perm[pos] : -1;
    f32x2 nq[D];                                   // (-q_j, -q_j): c - q = c + (-q), as in grid_join.cu
#pragma unroll
    for (int j = 0; j < D; ++j) {
        const float qj = valid ? __ldg(p.Xp + static_cast<size_t>(my_id) * kRowFloats + pl->feat[j]) : 0.f;
        nq[j] = pack2(-qj, -qj);
    }

    // every candidate but the query itself (by index, reading A4): fn(key)
    auto stream = [&](auto&& fn) {
        const int n_pairs = (N + 1) >> 1;
        constexpr int kTilePairs = kTileB / 2;
        constexpr int PF = (kTilePairs * G4 + 31) / 32;      // float4 per lane per tile
        float4 nx[PF];                                       // the next tile, in flight while this one is evaluated
        int nid0 = -1, nid1 = -1;
        auto fetch = [&](int t0) {
            const int n4 = min(kTilePairs, n_pairs - t0) * G4;
            const float4* src = reinterpret_cast<const float4*>(p.Xs) + static_cast<size_t>(t0) * G4;
#pragma unroll
            for (int u = 0; u < PF; ++u)
                if (lane + 32 * u < n4) nx[u] = __ldg(src + lane + 32 * u);
            nid0 = 2 * t0 + lane < N ? __ldg(p.perm + 2 * t0 + lane) : -1;
            nid1 = 2 * t0 + 32 + lane < N ? __ldg(p.perm + 2 * t0 + 32 + lane) : -1;
        };
        if (warp * kTilePairs < n_pairs) fetch(warp * kTilePairs);
        for (int t0 = warp * kTilePairs; t0 < n_pairs; t0 += kWarpsB * kTilePairs) {
            const int n = min(kTilePairs, n_pairs - t0);
            __syncwarp();
#pragma unroll
            for (int u = 0; u < PF; ++u)
                if (lane + 32 * u < n * G4) tile4[lane + 32 * u] = nx[u];
            tile_id[lane] = nid0;
            tile_id[32 + lane] = nid1;
            __syncwarp();
            if (t0 + kWarpsB * kTilePairs < n_pairs) fetch(t0 + kWarpsB * kTilePairs);
#pragma unroll 2
            for (int r = 0; r < n; ++r) {
                f32x2 acc = 0ull;
#pragma unroll
                for (int g = 0; g < G4; ++g) {
                    const float4 v = tile4[r * G4 + g];
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
                const int c0 = 2 * (t0 + r);
                const int id0 = tile_id[2 * r], id1 = tile_id[2 * r + 1];
                if (valid && c0 != pos) fn((static_cast<u64>(__float_as_uint(a0)) << kIdBits) | static_cast<u64>(id0));
                if (valid && c0 + 1 != pos && id1 >= 0)
                    fn((static_cast<u64>(__float_as_uint(a1)) << kIdBits) | static_cast<u64>(id1));
            }
        }
        __syncwarp();
    };

    // ---- radix selection of the k-th smallest key, 8 bits per pass from the top of the 48
    u64 prefix = 0;
    int need = k;
    bool done = !valid;            // the k-th key is pinned down as far as the emit pass needs
#pragma unroll 1
    for (int pass = 0; pass < 6; ++pass) {
        if (__all_sync(kFull, done)) break;       // the same in every warp of the CTA: they select identically
        const int shift = 40 - 8 * pass;
        __syncthreads();                           // the other warps have read this histogram
        for (int i = lane; i < kBins * 32; i += 32) hist[i] = 0;
        const u64 want = prefix >> (shift + 8);
        stream([&](u64 key) {
            if (!done && (pass == 0 || (key >> (shift + 8)) == want))
                hist[static_cast<unsigned>((key >> shift) & 255u) * 32 + lane] += 1;
        });
        __syncthreads();
        if (!done) {
            int cum = 0, sel = kBins - 1, csel = 0;
            bool found = false;
            for (int b = 0; b < kBins; ++b) {
                int c = 0;
#pragma unroll
                for (int w = 0; w < kWarpsB; ++w)
                    c += static_cast<int>(reinterpret_cast<const C*>(reinterpret_cast<const float*>(smem_raw) +
                                                                     static_cast<size_t>(w) * warp_words_b(D, sizeof(C)) +
                                                                     kTileB * DP + kTileB)[b * 32 + lane]);
                if (!found && cum + c >= need) { sel = b; csel = c; found = true; }
                if (!found) cum += c;
            }
            prefix |= static_cast<u64>(sel) << shift;
            need -= cum;
            // the k-th is the last of its bin: every key with this prefix is among the k smallest, the lower bits
            // need not be resolved (the usual case once the bins are narrower than the gaps between distances)
            if (found && need == csel) {
                prefix |= (static_cast<u64>(1) << shift) - 1;
                done = true;
            }
        }
    }
    // ---- the k keys up to the k-th, in stream order
    if (warp == 0) emit_cnt[lane] = 0;
    __syncthreads();
    u64* mine = keys_out + static_cast<size_t>(valid ? my_id - p.q_begin : 0) * k;
    stream([&](u64 key) {
        if (key <= prefix) {
            const int at = atomicAdd(&emit_cnt[lane], 1);    // any order: the segments are sorted afterwards
            if (at < k) mine[at] = key;
        }
    });
}

__global__ void offsets_kernel(int* __restrict__ off, int nq, int k) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i <= nq; i += gridDim.x * blockDim.x) off[i] = i * k;
}

// lists: one thread per entry
__global__ void bigk_lists_kernel(const u64* __restrict__ keys, long long total, int32_t* __restrict__ out_idx,
                                  float* __restrict__ out_dist, int32_t* __restrict__ out_indeg) {
    for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < total;
         i += static_cast<long long>(gridDim.x) * blockDim.x) {
        const u64 key = keys[i];
        const int id = static_cast<int>(key & ((1u << kIdBits) - 1u));
        if (out_idx) out_idx[i] = id;
        if (out_dist) out_dist[i] = sqrtf(__uint_as_float(static_cast<unsigned>(key >> kIdBits)));
        if (out_indeg) atomicAdd(&out_indeg[id], 1);
    }
}

// scores: one warp per query would reorder the sum; one thread per query keeps the list order of the other paths
__global__ void bigk_scores_kernel(const u64* __restrict__ keys, int nq, int k, float* __restrict__ out_kth,
                                   float* __restrict__ out_mean) {
    for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < nq; q += gridDim.x * blockDim.x) {
        const u64* row = keys + static_cast<size_t>(q) * k;
        float s = 0.f, dk = 0.f;
        for (int e = 0; e < k; ++e) {
            const float dd = sqrtf(__uint_as_float(static_cast<unsigned>(row[e] >> kIdBits)));
            s += dd;
            dk = dd;
        }
        if (out_kth) out_kth[q] = dk;
        if (out_mean) out_mean[q] = s / static_cast<float>(k);
    }
}

size_t al256(size_t x) { return (x + 255) / 256 * 256; }

size_t cub_bytes_for(int64_t nq, int k) {
    size_t b = 0;
    cub::DeviceSegmentedRadixSort::SortKeys(nullptr, b, static_cast<const u64*>(nullptr), static_cast<u64*>(nullptr),
                                            static_cast<int>(nq * k), static_cast<int>(nq), static_cast<const int*>(nullptr),
                                            static_cast<const int*>(nullptr), 0, 48);
    return al256(b);
}

template <int D, typename C>
cudaError_t launch_dc(const GridJoinParams& p, u64* keys, cudaStream_t st) {
    const size_t smem = (static_cast<size_t>(kWarpsB) * warp_words_b(D, sizeof(C)) + 32) * 4;
    auto kernel = bigk_select_kernel<D, C>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    if (e != cudaSuccess) return e;
    const long long groups = (static_cast<long long>(p.nq) + 31) / 32;
    kernel<<<static_cast<int>(groups), kWarpsB * 32, smem, st>>>(p, keys);
    return cudaGetLastError();
}

template <int D>
cudaError_t launch_d(const GridJoinParams& p, u64* keys, cudaStream_t st) {
    return p.N < 65536 ? launch_dc<D, unsigned short>(p, keys, st) : launch_dc<D, unsigned>(p, keys, st);
}

}  // namespace

size_t knn_bigk_scratch_bytes(int64_t nq, int k) {
    const size_t n = static_cast<size_t>(nq) * static_cast<size_t>(k);
    return 2 * al256(n * 8) + al256((static_cast<size_t>(nq) + 1) * 4) + cub_bytes_for(nq, k);
}

cudaError_t knn_bigk_launch(const GridJoinParams& p, int d, void* scratch, size_t scratch_bytes, cudaStream_t st) {
    if (p.N > kBigKMaxN || p.k < 1 || static_cast<long long>(p.nq) * p.k > 0x7fffffffLL) return cudaErrorInvalidValue;
    if (scratch_bytes < knn_bigk_scratch_bytes(p.nq, p.k)) return cudaErrorInvalidValue;
    const size_t n = static_cast<size_t>(p.nq) * static_cast<size_t>(p.k);
    unsigned char* r = static_cast<unsigned char*>(scratch);
    u64* keys_a = reinterpret_cast<u64*>(r); r += al256(n * 8);
    u64* keys_b = reinterpret_cast<u64*>(r); r += al256(n * 8);
    int* off = reinterpret_cast<int*>(r); r += al256((static_cast<size_t>(p.nq) + 1) * 4);
    size_t cub_bytes = cub_bytes_for(p.nq, p.k);
    cudaError_t e = cudaSuccess;
    switch (d) {
        case 1: e = launch_d<1>(p, keys_a, st); break;
        case 2: e = launch_d<2>(p, keys_a, st); break;
        case 3: e = launch_d<3>(p, keys_a, st); break;
        case 4: e = launch_d<4>(p, keys_a, st); break;
        case 5: e = launch_d<5>(p, keys_a, st); break;
        case 6: e = launch_d<6>(p, keys_a, st); break;
        case 7: e = launch_d<7>(p, keys_a, st); break;
        case 8: e = launch_d<8>(p, keys_a, st); break;
        case 9: e = launch_d<9>(p, keys_a, st); break;
        case 10: e = launch_d<10>(p, keys_a, st); break;
        case 11: e = launch_d<11>(p, keys_a, st); break;
        case 12: e = launch_d<12>(p, keys_a, st); break;
        case 13: e = launch_d<13>(p, keys_a, st); break;
        case 14: e = launch_d<14>(p, keys_a, st); break;
        case 15: e = launch_d<15>(p, keys_a, st); break;
        default: return cudaErrorInvalidValue;
    }
    if (e != cudaSuccess) return e;
    offsets_kernel<<<64, 256, 0, st>>>(off, p.nq, p.k);
    e = cub::DeviceSegmentedRadixSort::SortKeys(r, cub_bytes, keys_a, keys_b, static_cast<int>(n), p.nq, off, off + 1, 0, 48, st);
    if (e != cudaSuccess) return e;
    bigk_lists_kernel<<<148 * 8, 256, 0, st>>>(keys_b, static_cast<long long>(n), p.out_idx, p.out_dist, p.out_indeg);
    if (p.out_kth || p.out_mean)
        bigk_scores_kernel<<<(p.nq + 127) / 128, 128, 0, st>>>(keys_b, p.nq, p.k, p.out_kth, p.out_mean);
    return cudaGetLastError();
}

}  // namespace snaps
