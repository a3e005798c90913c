// range_lattice.cuh -- launch interface of the sub-lattice eps range self-join kernel.
#pragma once
#include "snaps_device.cuh"

namespace snaps {

constexpr int kRangeMaxThreads = 512;

struct RangeParams {
    const float* Xp;            // staged table, row-major (query rows)
    const float4* Xb;           // staged table, blocked (candidate stream)
    int n_blocks;               // ceil(N / 32)
    int N;
    int q_begin;                // queries are the objects q_begin .. q_begin + nq - 1
    int nq;
    const BatchDesc* batches;   // thr[] = nextafter(eps^2) per slot, -1 for unused slots
    int n_batches;
    int batches_per_item;
    int n_bchunks;
    int warps;                  // warps per CTA (each works on its own query)
    unsigned long long* work_counter;  // device, zeroed before launch
    uint32_t* out_count;        // [n_masks][nq]
    float* out_sum;
    float* out_mean;
};

size_t range_lattice_smem_bytes(int warps);
cudaError_t range_lattice_launch(const RangeParams& p, int grid, cudaStream_t stream);

}  // namespace snaps
