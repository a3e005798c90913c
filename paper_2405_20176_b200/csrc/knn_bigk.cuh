// knn_bigk.cuh -- kNN self-join of one feature subspace for long lists on small tables
// (384 < k <= 4096, N <= 131,072: the paper's k_max = 4096 on SNAPShot1).
#pragma once
#include "grid_join.cuh"

namespace snaps {

constexpr int kBigKMaxN = 1 << 17;     // ids take 17 bits of the 48-bit selection key
constexpr int kBigKMinK = 385;         // below, the heaps of grid_join.cu are faster for most masks (measured at N = 31,693:
                                       // k = 400: heaps 14-40 ms for d = 2 ... 15, selection 23-28 ms; k = 300: 10-32 ms)

// Whether the selection path beats the heaps: its passes cost ~N^2, the heaps ~N k log k.  Measured crossovers
// (join kernels, d = 2 ... 15): N = 31,693 k ~ 350; N = 65,000 k ~ 400; N = 131,072 k ~ 800 (heaps 97-192 ms at k = 400,
// selection 300-440 ms; at k = 1,024 480-550 against 310-470 ms).
inline bool knn_bigk_pays(int64_t N, int k) { return k >= kBigKMinK && N <= kBigKMaxN && 160LL * k >= N; }

// Scratch the launch needs for nq queries and lists of k: two arrays of nq*k 64-bit keys, segment offsets, CUB's own.
size_t knn_bigk_scratch_bytes(int64_t nq, int k);

// Same inputs and outputs as grid_knn_launch (the index of grid_index.cu supplies the compact rows and the
// sorted order; the cells themselves are not used).  The distances are formed by the same instruction sequence,
// so the two paths give identical lists.
cudaError_t knn_bigk_launch(const GridJoinParams& p, int d, void* scratch, size_t scratch_bytes, cudaStream_t stream);

}  // namespace snaps
