// ranking.cu -- NEXT-1: ranking function R, top-n overlap f (Eq. 2), parameter selection (Eq. 3)
// and k-grid prefix scores, on the device (the paper does these on the CPU in Python and names them
// its bottleneck on SNAPShot1).
//
//   R: rank 0 = most outlying, equal scores share a rank, ranks are dense (Table 2).
//   Which end is outlying: fewest neighbours / lowest in-degree, largest mean
//   distance; an object without eps-neighbours ranks first.
//   top-n = the first n objects of the stable order by (outlyingness, id) (reading A15).
#include "ranking.cuh"

#include <cub/device/device_segmented_radix_sort.cuh>

namespace snaps {

// Sort key: ascending uint32 = most outlying first.
__global__ void rank_keys_kernel(int metric, const void* __restrict__ values,
                                 const uint32_t* __restrict__ counts, int64_t N, int64_t total,
                                 uint32_t* __restrict__ keys, int32_t* __restrict__ ids) {
    for (int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; i < total;
         i += static_cast<int64_t>(gridDim.x) * blockDim.x) {
        uint32_t key;
        if (metric == 0 || metric == 2) {
            key = static_cast<const uint32_t*>(values)[i];             // small is outlying
        } else {
            // large is outlying: non-negative floats order like their bit patterns; invert
            key = ~__float_as_uint(static_cast<const float*>(values)[i]);
            if (metric == 1 && counts[i] == 0) key = 0u;               // no neighbours: first
        }
        keys[i] = key;
        ids[i] = static_cast<int32_t>(i % N);
    }
}

// One CTA per row: dense ranks from the sorted keys (rank = number of key changes before p).
__global__ void dense_rank_kernel(const uint32_t* __restrict__ keys_sorted,
                                  const int32_t* __restrict__ order, int64_t N,
                                  int32_t* __restrict__ out_rank) {
    __shared__ int s_warp[32];
    __shared__ int s_carry;
    const int64_t row = blockIdx.x;
    const uint32_t* k = keys_sorted + row * N;
    const int32_t* o = order + row * N;
    int32_t* r = out_rank + row * N;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int64_t base = 0; base < N; base += blockDim.x) {
        const int64_t p = base + threadIdx.x;
        int flag = (p < N && p > 0 && k[p] != k[p - 1]) ? 1 : 0;
        int incl = flag;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += v;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            int w = lane < nw ? s_warp[lane] : 0;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int v = __shfl_up_sync(0xffffffffu, w, d);
                if (lane >= d) w += v;
            }
            s_warp[lane] = w;   // inclusive over warps
        }
        __syncthreads();
        const int before = s_carry + (warp > 0 ? s_warp[warp - 1] : 0) + incl;
        if (p < N) r[o[p]] = before;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) s_carry = before;
        __syncthreads();
    }
}

size_t rank_workspace_bytes(int64_t N, int n_rows) {
    const size_t total = static_cast<size_t>(N) * n_rows;
    size_t cub_bytes = 0;
    cub::DeviceSegmentedRadixSort::SortPairs(nullptr, cub_bytes, static_cast<const uint32_t*>(nullptr),
                                             static_cast<uint32_t*>(nullptr), static_cast<const int32_t*>(nullptr),
                                             static_cast<int32_t*>(nullptr), static_cast<int64_t>(total), n_rows,
                                             static_cast<const int64_t*>(nullptr), static_cast<const int64_t*>(nullptr));
    auto al = [](size_t x) { return (x + 255) / 256 * 256; };
    // keys in, keys out, ids in, ids out (when the caller does not want the order), offsets, cub
    return 4 * al(total * 4) + al((static_cast<size_t>(n_rows) + 1) * 8) + al(cub_bytes);
}

__global__ void row_offsets_kernel(int64_t N, int n_rows, int64_t* off) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i <= n_rows; i += gridDim.x * blockDim.x)
        off[i] = static_cast<int64_t>(i) * N;
}

cudaError_t rank_launch(int metric, const void* values, const uint32_t* counts, int64_t N, int n_rows,
                        int32_t* out_rank, int32_t* out_order, void* ws, size_t ws_bytes,
                        cudaStream_t stream) {
    if (ws_bytes < rank_workspace_bytes(N, n_rows)) return cudaErrorInvalidValue;
    const size_t total = static_cast<size_t>(N) * n_rows;
    auto al = [](size_t x) { return (x + 255) / 256 * 256; };
    unsigned char* p = static_cast<unsigned char*>(ws);
    uint32_t* keys_in = reinterpret_cast<uint32_t*>(p);
    uint32_t* keys_out = reinterpret_cast<uint32_t*>(p + al(total * 4));
    int32_t* ids_in = reinterpret_cast<int32_t*>(p + 2 * al(total * 4));
    int32_t* ids_tmp = reinterpret_cast<int32_t*>(p + 3 * al(total * 4));
    int64_t* off = reinterpret_cast<int64_t*>(p + 4 * al(total * 4));
    void* cub_tmp = p + 4 * al(total * 4) + al((static_cast<size_t>(n_rows) + 1) * 8);
    size_t cub_bytes = ws_bytes - (4 * al(total * 4) + al((static_cast<size_t>(n_rows) + 1) * 8));
    int32_t* order = out_order ? out_order : ids_tmp;
    const int grid = 148 * 8;
    rank_keys_kernel<<<grid, 256, 0, stream>>>(metric, values, counts, N, static_cast<int64_t>(total), keys_in, ids_in);
    row_offsets_kernel<<<(n_rows + 256) / 256, 256, 0, stream>>>(N, n_rows, off);
    // LSD radix sort is stable: equal keys keep increasing id order
    cudaError_t e = cub::DeviceSegmentedRadixSort::SortPairs(cub_tmp, cub_bytes, keys_in, keys_out, ids_in, order,
                                                             static_cast<int64_t>(total), n_rows, off, off + 1, 0, 32,
                                                             stream);
    if (e != cudaSuccess) return e;
    if (out_rank) dense_rank_kernel<<<n_rows, 256, 0, stream>>>(keys_out, order, N, out_rank);
    return cudaGetLastError();
}

// Eq. 2: one CTA per row pair; a bitmap of A's top-n in shared memory, B's top-n probes it.
// Row r of the output compares row r * stride_a + off_a of order_a with row r * stride_b + off_b of order_b.
__global__ void topn_overlap_kernel(const int32_t* __restrict__ order_a, const int32_t* __restrict__ order_b,
                                    int64_t N, int n, int stride_a, int off_a, int stride_b, int off_b,
                                    float* __restrict__ out_f) {
    extern __shared__ uint32_t bits[];
    __shared__ int s_hits;
    const int64_t row = blockIdx.x;
    order_a += (row * stride_a + off_a) * N;
    order_b += (row * stride_b + off_b) * N;
    const int words = static_cast<int>((N + 31) / 32);
    for (int i = threadIdx.x; i < words; i += blockDim.x) bits[i] = 0u;
    if (threadIdx.x == 0) s_hits = 0;
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const int id = order_a[i];
        atomicOr(&bits[id >> 5], 1u << (id & 31));
    }
    __syncthreads();
    int hits = 0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const int id = order_b[i];
        hits += (bits[id >> 5] >> (id & 31)) & 1u;
    }
    atomicAdd(&s_hits, hits);
    __syncthreads();
    if (threadIdx.x == 0) out_f[row] = static_cast<float>(s_hits) / static_cast<float>(n);
}

cudaError_t topn_overlap_strided_launch(const int32_t* order_a, const int32_t* order_b, int64_t N, int n_rows, int n,
                                        int stride_a, int off_a, int stride_b, int off_b, float* out_f,
                                        cudaStream_t stream) {
    const size_t smem = static_cast<size_t>((N + 31) / 32) * 4;
    cudaError_t e = cudaFuncSetAttribute(topn_overlap_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(smem));
    if (e != cudaSuccess) return e;
    topn_overlap_kernel<<<n_rows, 256, smem, stream>>>(order_a, order_b, N, n, stride_a, off_a, stride_b, off_b, out_f);
    return cudaGetLastError();
}

cudaError_t topn_overlap_launch(const int32_t* order_a, const int32_t* order_b, int64_t N, int n_rows, int n,
                                float* out_f, cudaStream_t stream) {
    return topn_overlap_strided_launch(order_a, order_b, N, n_rows, n, 1, 0, 1, 0, out_f, stream);
}

// Eq. 3 per row: argmin_j |U_min[j] - U_max[j]| (first minimiser).  u_*: [G][n_rows].
// With n_top > 0 the fractions are taken back to integer hit counts (f = hits / n), so that equal
// differences compare equal and the first minimiser is well defined.
__global__ void select_kernel(const float* __restrict__ u_min, const float* __restrict__ u_max, int G,
                              int n_rows, int n_top, int32_t* __restrict__ out_j) {
    const float sc = n_top > 0 ? static_cast<float>(n_top) : 1.f;
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < n_rows; r += gridDim.x * blockDim.x) {
        int best = 0;
        float bd = fabsf(n_top > 0 ? rintf(u_min[r] * sc) - rintf(u_max[r] * sc) : u_min[r] - u_max[r]);
        for (int j = 1; j < G; ++j) {
            const float a = u_min[static_cast<size_t>(j) * n_rows + r], b = u_max[static_cast<size_t>(j) * n_rows + r];
            const float d = fabsf(n_top > 0 ? rintf(a * sc) - rintf(b * sc) : a - b);
            if (d < bd) {
                bd = d;
                best = j;
            }
        }
        out_j[r] = best;
    }
}

cudaError_t select_launch(const float* u_min, const float* u_max, int G, int n_rows, int n_top, int32_t* out_j,
                          cudaStream_t stream) {
    select_kernel<<<(n_rows + 255) / 256, 256, 0, stream>>>(u_min, u_max, G, n_rows, n_top, out_j);
    return cudaGetLastError();
}

// the k_max lists contain the lists of every k_j < k_max (their first k_j entries).
__global__ void scores_at_k_kernel(int64_t N, int n_masks, int k_max, int kj, const int32_t* __restrict__ idx,
                                   const float* __restrict__ dist, float* __restrict__ out_kth,
                                   float* __restrict__ out_mean, int32_t* __restrict__ out_indeg) {
    const int64_t total = N * n_masks;
    for (int64_t o = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; o < total;
         o += static_cast<int64_t>(gridDim.x) * blockDim.x) {
        const int64_t m = o / N;
        if (dist) {
            float sum = 0.f, dk = 0.f;
            for (int e = 0; e < kj; ++e) {
                dk = dist[o * k_max + e];
                sum += dk;
            }
            if (out_kth) out_kth[o] = dk;
            if (out_mean) out_mean[o] = sum / static_cast<float>(kj);
        }
        if (idx && out_indeg)
            for (int e = 0; e < kj; ++e) atomicAdd(&out_indeg[m * N + idx[o * k_max + e]], 1);
    }
}

cudaError_t scores_at_k_launch(int64_t N, int n_masks, int k_max, int kj, const int32_t* idx, const float* dist,
                               float* out_kth, float* out_mean, int32_t* out_indeg, cudaStream_t stream) {
    const int64_t total = N * n_masks;
    const int grid = static_cast<int>(total / 256 + 1 < 148 * 32 ? total / 256 + 1 : 148 * 32);
    scores_at_k_kernel<<<grid, 256, 0, stream>>>(N, n_masks, k_max, kj, idx, dist, out_kth, out_mean, out_indeg);
    return cudaGetLastError();
}

}  // namespace snaps
