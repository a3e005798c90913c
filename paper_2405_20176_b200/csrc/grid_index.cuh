// grid_index.cuh -- the per-subspace grid index of the large-N / arbitrary-mask engine.
//
// PAPER.md:297 (section 3.8.1): the paper's joins index c <= 6 of a feature space's dimensions
// with a grid and refine by distance calculations.  Here: per table,
// every feature gets 4096 equi-depth ("quantile") master bins; per mask, up to three of its
// features -- the ones with the most spread-out distributions -- are binned at a resolution that
// leaves ~16 objects per cell, objects are sorted by cell, and the mask's columns are gathered
// into compact rows in cell order.  The join kernels (grid_join.cuh) then walk the cells around a
// group of 32 neighbouring queries with exact per-cell lower bounds.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "snaps_device.cuh"

namespace snaps {

constexpr int kGridMasterBits = 12;
constexpr int kGridMaster = 1 << kGridMasterBits;       // master bins per feature
constexpr int kGridEdgeStride = kGridMaster + 1;        // edges per feature (last = column maximum)
constexpr int kGridDims = 3;                            // grid dimensions (leading ones may be unused)
constexpr int kGridSlackRows = 64;                      // spare rows at the end of the compact table (odd N: the last pair's partner)

// Per mask, written by grid_plan_kernel on the device (the choice of index features depends on the
// data) except d / bits, which the host fixes from popcount(mask) and N.
struct GridPlan {
    int32_t d;                 // features of the mask
    int32_t feat[15];          // the mask's features, ascending: column j of the compact rows = feat[j]
    int32_t idx_feat[kGridDims];   // index feature of grid dimension g (ascending in g), -1 = unused
    int32_t idx_col[kGridDims];    // its column in the compact row
    int32_t bits[kGridDims];       // log2(bins) of dimension g (0 for unused dimensions)
    int32_t pad_;
};

struct GridTable {             // per-table state inside the workspace
    const float* Xp;           // staged rows (80 B)
    float* edges;              // [15][kGridEdgeStride] master bin edges (ascending)
    uint16_t* bin12;           // [15][n_pad] master bin of every object
    float* score;              // [15] concentration of each feature (lower = better index feature)
    int* iota;                 // [n_pad] 0,1,2,...
    int n_pad;
};

struct GridIndex {             // per-mask state (rebuilt for every mask)
    uint32_t* keys_in;
    uint32_t* keys;            // sorted cell keys [N]
    int* perm;                 // sorted position -> object id
    int* cell_start;           // [n_cells + 1]
    float* Xs;                 // compact rows in cell order, two objects interleaved: [ceil(N/2)][4*ceil(d/4)][2] floats
    int* qlist;                // positions of the queries in [q_begin, q_end) (only when sharded)
    int* warp_order;           // kNN: the join's warps (32 consecutive queries each), heaviest first
    void* cub_tmp;
    size_t cub_bytes;
};

// log2(bins) per grid dimension for a mask of d features on N objects (host and device agree).
__host__ __device__ inline void grid_bits_for(int64_t N, int d, int bits[kGridDims]) {
    const int c = d < kGridDims ? d : kGridDims;
    // ~16 objects per cell: total bits = log2(N / 16), split evenly over the c dimensions
    int total = 0;
    while ((static_cast<int64_t>(16) << (total + 1)) <= N) ++total;
    int per = total / c;
    if (per > kGridMasterBits) per = kGridMasterBits;
    if (per < 1) per = 1;
    for (int g = 0; g < kGridDims; ++g) bits[g] = (g >= kGridDims - c) ? per : 0;
}

size_t grid_table_bytes(int64_t N);
size_t grid_index_bytes(int64_t N);

// One-time per call: master edges, master bins of every object, feature scores, iota.
// `scratch` is the (not yet used) per-mask index region.
cudaError_t grid_table_build(const float* Xp, int N, int n_feat, GridTable* t, unsigned char* table_region,
                             unsigned char* index_region, size_t index_bytes, cudaStream_t stream);

// Plans for all masks (device masks -> device plans).
cudaError_t grid_plan_launch(const uint16_t* d_masks, int n_masks, int64_t N, const GridTable& t,
                             GridPlan* d_plans, cudaStream_t stream);

void grid_index_carve(unsigned char* region, size_t bytes, int64_t N, GridIndex* ix);

// Per mask: cell keys -> stable sort -> compact rows, cell starts; optional query list for [q_begin, q_end).
// knn_k > 0: also the order in which the kNN join takes its warps (ix->warp_order), heaviest first.
cudaError_t grid_index_build(const GridTable& t, const GridPlan* d_plan, int N, int d, const int bits[kGridDims],
                             int64_t q_begin, int64_t q_end, int knn_k, GridIndex* ix, cudaStream_t stream);

}  // namespace snaps
