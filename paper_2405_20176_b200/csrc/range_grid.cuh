// range_grid.cuh -- launch interface of the radius-grid eps range self-join kernel.
#pragma once
#include "snaps_device.cuh"

namespace snaps {

constexpr int kRangeGridMaxThreads = 512;
constexpr int kRangeGridMaxRadii = 32;

struct RangeGridParams {
    const float* Xp;
    const float4* Xb;
    int n_blocks;
    int N;
    int q_begin;                // queries are the objects q_begin .. q_begin + nq - 1
    int nq;
    int G;                      // radii per mask, ascending
    const BatchDesc* batches;   // slot[] only (thr[] unused)
    int n_batches;
    const float* thr_grid;      // device [n_masks][G]: nextafter(eps^2)
    int warps;
    unsigned long long* work_counter;
    uint32_t* out_count;        // [n_masks][G][nq]
    float* out_sum;
    float* out_mean;
};

size_t range_grid_smem_bytes(int G, int warps);
cudaError_t range_grid_launch(const RangeGridParams& p, int grid, cudaStream_t stream);

}  // namespace snaps
