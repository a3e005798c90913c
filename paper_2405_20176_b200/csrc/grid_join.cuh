// grid_join.cuh -- launch interface of the grid-engine joins (one mask per launch).
#pragma once
#include "grid_index.cuh"

namespace snaps {

constexpr int kGridMaxK = 256;          // kNN lists up to this length live in shared memory (k_max = 256 on LSST5M)
constexpr int kGridMaxKBig = 4096;      // beyond it the heaps live in the output lists (k_max = 4096 on SNAPShot1)

struct GridJoinParams {
    // index of this mask (grid_index.cuh)
    const float* Xp;           // staged rows (query coordinates)
    const float* Xs;           // compact pair-interleaved rows in cell order
    const uint32_t* keys;
    const int* perm;
    const int* cell_start;
    const int* qlist;          // sorted positions of the queries, or nullptr = every position
    const int* warp_order;     // warp slot -> group of 32 queries (heaviest first), or nullptr = identity
    const float* edges;        // [15][kGridEdgeStride]
    const GridPlan* plan;      // device
    int bits[kGridDims];       // host copy of plan->bits
    int N;
    int nq;                    // number of queries (q_end - q_begin)
    int q_begin;
    // kNN (outputs of this mask: rows of nq entries, in-degree row of N entries)
    int k;
    int32_t* out_idx;
    float* out_dist;
    float* out_kth;
    float* out_mean;
    int32_t* out_indeg;
    // range join
    float eps2;                // fl(eps^2): a pair is a neighbour iff d^2 <= eps2 (closed ball, reading A2)
    uint32_t* out_count;
    float* out_sum;
    float* out_rmean;
    // radius grid (range join at G ascending radii): thresholds on the device
    int G;
    const float* eps2_grid;    // [G] fl(eps_g^2) ascending (this mask's row)
};

cudaError_t grid_knn_launch(const GridJoinParams& p, int d, cudaStream_t stream);
cudaError_t grid_range_launch(const GridJoinParams& p, int d, cudaStream_t stream);

}  // namespace snaps
