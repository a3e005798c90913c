// knn_lattice.cuh -- launch interface of the sub-lattice kNN self-join kernel.
#pragma once
#include "snaps_device.cuh"

namespace snaps {

constexpr int kKnnMaxThreads = 512;  // 16 warps x 128 registers
constexpr int kLatticeMaxK = 32;     // list length the sub-lattice kernel holds in shared memory

struct KnnParams {
    const float* Xp;            // staged table, row-major, n_tiles*128 rows of 20 floats (seeds, query rows)
    const float4* Xb;           // staged table, blocked: [n_blocks][4 feature groups][32 rows] float4
    int n_blocks;               // ceil(N / 32)
    int N;
    int q_begin;                // queries are the objects q_begin .. q_begin + nq - 1
    int nq;
    int k;
    const BatchDesc* batches;   // device
    int n_batches;
    int batches_per_item;       // consecutive batches one warp keeps its query for
    int n_bchunks;              // ceil(n_batches / batches_per_item)
    int warps;                  // warps per CTA (each works on its own query)
    unsigned long long* work_counter;  // device, zeroed before launch
    int32_t* out_idx;           // [n_masks][nq][k]
    float* out_dist;
    float* out_kth;             // [n_masks][nq]
    float* out_mean;
    int32_t* out_indeg;         // [n_masks][N]
};

size_t knn_lattice_smem_bytes(int k, int warps);
cudaError_t knn_lattice_launch(const KnnParams& p, int grid, cudaStream_t stream);

}  // namespace snaps
