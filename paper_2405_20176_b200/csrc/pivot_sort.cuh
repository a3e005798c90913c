// pivot_sort.cuh -- per-feature sorted copies of the table for the pivot sweep (large-N kNN path).
#pragma once
#include "snaps_device.cuh"

namespace snaps {

// Device scratch pivot_build needs for a table of n_pad rows.
size_t pivot_sort_temp_bytes(int n_pad);

// Sort the staged rows (Xp, 20 floats per row, n_pad rows incl. padding) by feature f.
//   Xs     [n_pad/32][4][32] float4 : blocked table in sorted order
//   piv    [n_pad]  sorted values of feature f
//   idmap  [n_pad]  sorted position -> row index (object id; >= N for padding rows)
//   pos    [N]      object id -> sorted position
cudaError_t pivot_build(const float* Xp, int N, int n_pad, int f, float4* Xs, float* piv, int* idmap,
                        int* pos, void* temp, size_t temp_bytes, cudaStream_t stream);

}  // namespace snaps
