// snaps_device.cuh -- device-side building blocks shared by the join kernels (sm_100a).
//
// Layout of the staged table ("a1" in DESIGN.md): row r of the caller's N x n_feat
// fp32 matrix becomes 20 floats (80 bytes): features 0..14, then 5 zeros.  80 B
// rows make per-lane 128-bit shared-memory reads conflict-free (lane stride 20
// words -> the 8 lanes of a quarter-warp hit 8 disjoint 4-bank groups) and keep
// a tile of rows one contiguous block, so a tile moves with ONE bulk async copy
// (cp.async.bulk, SASS UBLKCP) that signals an mbarrier.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace snaps {

constexpr int kRowFloats = 20;                 // staged row: 15 features + 5 pad
constexpr int kRowBytes = kRowFloats * 4;      // 80
constexpr int kTileRows = 128;                 // candidates per smem tile
constexpr int kTileBytes = kTileRows * kRowBytes;  // 10240
constexpr int kStages = 3;                     // tile ring depth
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

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t"
        "}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// 1-D bulk async copy global -> shared, completion counted in bytes on `bar`.
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, uint32_t bytes,
                                         uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(smem_u32(smem_dst)),
        "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

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
