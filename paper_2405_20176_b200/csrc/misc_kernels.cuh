// misc_kernels.cuh -- table staging (a1), standalone score kernels (a7), FP32 rate probes.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace snaps {

cudaError_t stage_table_launch(const float* X, int64_t ld, int N, int n_feat, float* Xp,
                               int n_rows_padded, cudaStream_t stream);

cudaError_t stage_blocked_launch(const float* X, int64_t ld, int N, int n_feat, float4* Xb,
                                 int n_blocks, cudaStream_t stream);

cudaError_t knn_scores_launch(int64_t N, int n_masks, int k, const int32_t* idx, const float* dist,
                              float* out_kth, float* out_mean, int32_t* out_indeg,
                              cudaStream_t stream);

cudaError_t eps_mean_launch(int64_t total, const uint32_t* cnt, const float* sum, float* out_mean,
                            cudaStream_t stream);

cudaError_t range_from_knn_launch(int64_t nq, int n_masks, int k, const float* dist, const float* d_eps,
                                  uint32_t* out_count, float* out_sum, float* out_mean, uint8_t* out_complete,
                                  cudaStream_t stream);

// kind 0: FFMA, 1: FADD, 2: FADD+FSETP pairs.  Returns lane-ops executed and elapsed ms.
cudaError_t probe_fp32_launch(int kind, double* lane_ops, float* ms, float* d_scratch, cudaStream_t stream);

}  // namespace snaps
