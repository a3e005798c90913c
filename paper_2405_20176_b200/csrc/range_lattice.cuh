// range_lattice.cuh -- launch interface of the sub-lattice eps range self-join kernel.
#pragma once
#include "snaps_device.cuh"

namespace snaps {

constexpr int kRangeMaxThreads = 512;

struct RangeParams {
    const float* Xp;            // staged table, row-major (query rows)
    const float4* Xb;           // staged table, blocked (candidate stream)
    int n_blocks;               // ceil(N / 32)
    int sweep;                  // 1: pivot sweep over the sorted copies below (pivot_sort.cuh)
    const float4* Xs[15];
    const float* piv[15];
    const int* idmap[15];
    const int* pos[15];
    int N;
    const BatchDesc* batches;   // thr[] = nextafter(eps^2) per slot, -1 for unused slots
    int n_batches;
    int batches_per_item;
    int n_bchunks;
    int warps;                  // warps per CTA (each works on its own query)
    unsigned long long* work_counter;  // device, zeroed before launch
    uint32_t* out_count;
    float* out_sum;
    float* out_mean;
};

size_t range_lattice_smem_bytes(int warps);
cudaError_t range_lattice_launch(const RangeParams& p, int grid, cudaStream_t stream);

}  // namespace snaps
