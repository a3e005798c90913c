// eps_search.cuh -- NEXT-2: sampled distance histogram per mask (device part of the eps search).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace snaps {

size_t dist_hist_workspace_bytes(int nq, int nc, int n_masks);
cudaError_t dist_hist_launch(const float* X, int64_t ld, int n_feat, const int32_t* h_q, int nq, const int32_t* h_c,
                             int nc, const uint16_t* h_masks, const float* h_rmax, int n_masks, int n_bins,
                             unsigned long long* out_hist, void* ws, cudaStream_t st);


// The whole search on the device: eps_mean per mask (mean sampled distance), the histogram over
// [0, eps_mean), and the radius for each target selectivity.  pairs = sampled (q, c) pairs with c != q.
size_t eps_search_workspace_bytes(int nq, int nc, int n_masks, int n_bins, int n_targets);
cudaError_t eps_search_launch(const float* X, int64_t N, int64_t ld, int n_feat, const int32_t* h_q, int nq, const int32_t* h_c,
                              int nc, long long pairs, const uint16_t* h_masks, int n_masks, int n_bins,
                              const double* h_targets, int n_targets, float* out_eps_mean, float* out_eps,
                              unsigned long long* out_hist, void* ws, cudaStream_t st);


// G evenly spaced radii between eps_mm[m][0] and eps_mm[m][1] and their squared thresholds.
cudaError_t eps_grid_launch(const float* eps_mm, int n_masks, int G, int successor, float* eps_grid, float* thr,
                            cudaStream_t st);

}  // namespace snaps
