// pivot_sort.cu -- the pruning index of the large-N kNN path.
//
// For a batch whose masks all contain feature f (every mask of a batch contains the batch's high
// features H), an object c can enter a list of query q only if (x_cf - x_qf)^2 is below the
// batch's largest threshold.  With the table sorted by f, those objects are one contiguous run
// around q's own position, so the scan sweeps outwards from q and stops in each direction at the
// first block edge beyond the bound -- exact pruning, shared by the whole mask family.
// This file builds, per pivot feature: the blocked table in sorted order, the sorted pivot
// values, the position -> object id map and the object id -> position map.
#include "pivot_sort.cuh"

#include <cub/device/device_radix_sort.cuh>

namespace snaps {

__global__ void pivot_keys_kernel(const float* __restrict__ Xp, int n_pad, int f,
                                  uint32_t* __restrict__ keys, int* __restrict__ vals) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_pad; i += gridDim.x * blockDim.x) {
        // features are in [0,1] (padding rows 1e18): non-negative floats order like their bit patterns
        keys[i] = __float_as_uint(Xp[static_cast<size_t>(i) * kRowFloats + f]);
        vals[i] = i;
    }
}

__global__ void pivot_gather_kernel(const float* __restrict__ Xp, int N, int n_pad,
                                    const uint32_t* __restrict__ keys_sorted,
                                    const int* __restrict__ idmap, float4* __restrict__ Xs,
                                    float* __restrict__ piv, int* __restrict__ pos) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_pad; i += gridDim.x * blockDim.x) {
        const int r = idmap[i];
        piv[i] = __uint_as_float(keys_sorted[i]);
        if (r < N) pos[r] = i;
        const float4* row = reinterpret_cast<const float4*>(Xp + static_cast<size_t>(r) * kRowFloats);
        float4* dst = Xs + static_cast<size_t>(i >> 5) * 128 + (i & 31);
#pragma unroll
        for (int g = 0; g < 4; ++g) dst[g * 32] = row[g];
    }
}

size_t pivot_sort_temp_bytes(int n_pad) {
    size_t cub_bytes = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, cub_bytes, static_cast<const uint32_t*>(nullptr),
                                    static_cast<uint32_t*>(nullptr), static_cast<const int*>(nullptr),
                                    static_cast<int*>(nullptr), n_pad);
    const size_t arr = (static_cast<size_t>(n_pad) * 4 + 255) / 256 * 256;
    return 3 * arr + (cub_bytes + 255) / 256 * 256;   // keys in, keys out, values in, cub scratch
}

cudaError_t pivot_build(const float* Xp, int N, int n_pad, int f, float4* Xs, float* piv, int* idmap,
                        int* pos, void* temp, size_t temp_bytes, cudaStream_t stream) {
    const size_t arr = (static_cast<size_t>(n_pad) * 4 + 255) / 256 * 256;
    if (temp_bytes < pivot_sort_temp_bytes(n_pad)) return cudaErrorInvalidValue;
    unsigned char* t = static_cast<unsigned char*>(temp);
    uint32_t* keys_in = reinterpret_cast<uint32_t*>(t);
    uint32_t* keys_out = reinterpret_cast<uint32_t*>(t + arr);
    int* vals_in = reinterpret_cast<int*>(t + 2 * arr);
    void* cub_tmp = t + 3 * arr;
    size_t cub_bytes = temp_bytes - 3 * arr;
    const int grid = 148 * 8;
    pivot_keys_kernel<<<grid, 256, 0, stream>>>(Xp, n_pad, f, keys_in, vals_in);
    cudaError_t e = cub::DeviceRadixSort::SortPairs(cub_tmp, cub_bytes, keys_in, keys_out, vals_in, idmap,
                                                    n_pad, 0, 32, stream);
    if (e != cudaSuccess) return e;
    pivot_gather_kernel<<<grid, 256, 0, stream>>>(Xp, N, n_pad, keys_out, idmap, Xs, piv, pos);
    return cudaGetLastError();
}

}  // namespace snaps
