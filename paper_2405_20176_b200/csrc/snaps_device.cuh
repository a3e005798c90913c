// snaps_device.cuh -- device-side building blocks shared by the join kernels (sm_100a).
//
// Layouts of the staged table ("a1" in DESIGN.md).  Row-major copy Xp: row r of the caller's
// N x n_feat fp32 matrix becomes 20 floats (80 bytes): features 0..14, then 5 zeros; used for
// query rows, seed evaluations and as the gather source of the sorted copies.  Blocked copy Xb
// (the candidate stream of both join kernels): 32 rows per block, four feature groups of 32
// float4 per block, read with four fully coalesced 128-bit loads per warp.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace snaps {

constexpr int kRowFloats = 20;                 // staged row: 15 features + 5 pad
constexpr int kRowBytes = kRowFloats * 4;      // 80
constexpr int kTileRows = 128;                 // Xp is padded to a multiple of 128 rows
constexpr int kTileBytes = kTileRows * kRowBytes;  // 10240
constexpr int kLow = 6;                        // lattice features per batch
constexpr int kLat = 1 << kLow;                // 64 subset sums per (pair, batch)
constexpr int kRing = 128;                     // kNN: per-warp ring of (list, id, d^2) triples awaiting merge
constexpr unsigned kFull = 0xffffffffu;
constexpr float kPadCoord = 1e18f;             // coordinate of padding rows (squares stay finite: 15e36)

// One batch = the sub-lattice { H u T : T subset of features 0..5 } for a fixed
// set H of features 6..14 (all feature subsets are wanted, so
// complete sub-lattices are the common case).  slot[T] is the index of mask
// H|T in the caller's list, or -1 if that mask was not asked for.
struct alignas(16) BatchDesc {
    float thr[kLat];           // range join: nextafter(eps^2) per slot (unused for kNN); read as float4
    int32_t slot[kLat];
    uint32_t hmask;            // bits 6..14
    int32_t n_valid;
    int32_t pivot;             // pivot sweep: a feature every valid mask of the batch contains, or -1
    int32_t pad_;
};
static_assert(sizeof(BatchDesc) % 16 == 0, "BatchDesc rows are read with 128-bit loads");

// Squared distance on a runtime mask from two staged rows (slow paths only).
__device__ __forceinline__ float masked_d2(const float* __restrict__ a, const float* __restrict__ b,
                                           uint32_t mask) {
    float acc = 0.f;
#pragma unroll
    for (int j = 0; j < 15; ++j) {
        float diff = a[j] - b[j];
        float sq = __fmul_rn(diff, diff);
        if ((mask >> j) & 1u) acc = __fadd_rn(acc, sq);
    }
    return acc;
}

}  // namespace snaps
