// ranking.cuh -- NEXT-1 device steps: dense ranking, top-n overlap, parameter selection, k-grid scores.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace snaps {

size_t rank_workspace_bytes(int64_t N, int n_rows);
cudaError_t rank_launch(int metric, const void* values, const uint32_t* counts, int64_t N, int n_rows,
                        int32_t* out_rank, int32_t* out_order, void* ws, size_t ws_bytes, cudaStream_t stream);
cudaError_t topn_overlap_launch(const int32_t* order_a, const int32_t* order_b, int64_t N, int n_rows, int n,
                                float* out_f, cudaStream_t stream);
cudaError_t topn_overlap_strided_launch(const int32_t* order_a, const int32_t* order_b, int64_t N, int n_rows, int n,
                                        int stride_a, int off_a, int stride_b, int off_b, float* out_f,
                                        cudaStream_t stream);
cudaError_t select_launch(const float* u_min, const float* u_max, int G, int n_rows, int n_top, int32_t* out_j,
                          cudaStream_t stream);
cudaError_t scores_at_k_launch(int64_t N, int n_masks, int k_max, int kj, const int32_t* idx, const float* dist,
                               float* out_kth, float* out_mean, int32_t* out_indeg, cudaStream_t stream);

}  // namespace snaps
