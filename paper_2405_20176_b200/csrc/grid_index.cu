// grid_index.cu -- builds the grid index of grid_index.cuh (table-level quantile bins once per
// call, then per mask: cell keys, stable radix sort, compact rows in cell order, cell starts).
#include "grid_index.cuh"

#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_select.cuh>

namespace snaps {

namespace {

inline size_t al(size_t x) { return (x + 255) / 256 * 256; }
constexpr int kGrid = 148 * 8;

// order-preserving map float -> uint32 (negative values and -0.0 included)
__device__ __forceinline__ uint32_t f2key(float v) {
    const uint32_t b = __float_as_uint(v);
    return b ^ ((b >> 31) ? 0xffffffffu : 0x80000000u);
}
__device__ __forceinline__ float key2f(uint32_t k) {
    return __uint_as_float(k ^ ((k >> 31) ? 0x80000000u : 0xffffffffu));
}

__global__ void column_keys_kernel(const float* __restrict__ Xp, int N, int f, uint32_t* __restrict__ keys) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x)
        keys[i] = f2key(Xp[static_cast<size_t>(i) * kRowFloats + f]);
}

// master edges of one feature from its sorted values: edge b = value at rank floor(b N / 4096)
__global__ void edges_kernel(const uint32_t* __restrict__ sorted, int N, float* __restrict__ edges) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < kGridMaster) edges[b] = key2f(sorted[(static_cast<long long>(b) * N) >> kGridMasterBits]);
    if (b == kGridMaster) edges[b] = key2f(sorted[N - 1]);
}

// master bin of x: the last b with edges[b] <= x (edges[0] is the column minimum)
__device__ __forceinline__ int master_bin(const float* __restrict__ edges, float x) {
    int lo = 0, hi = kGridMaster;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (edges[mid] <= x) lo = mid + 1; else hi = mid;
    }
    return lo > 0 ? lo - 1 : 0;
}

__global__ void bins_kernel(const float* __restrict__ Xp, int N, int f, const float* __restrict__ edges,
                            uint16_t* __restrict__ bin12) {
    __shared__ float e[kGridMaster];
    for (int b = threadIdx.x; b < kGridMaster; b += blockDim.x) e[b] = edges[b];
    __syncthreads();
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x)
        bin12[i] = static_cast<uint16_t>(master_bin(e, Xp[static_cast<size_t>(i) * kRowFloats + f]));
}

// Concentration of a feature: sum over 64 equi-depth bins of 1 / width ~ integral of density^2.
// The mass a slab of half-width r around a query holds is ~ 2 r x this, so low = good index feature.
__global__ void score_kernel(const float* __restrict__ edges, int n_feat, float* __restrict__ score) {
    const int f = threadIdx.x;
    if (f >= 15) return;
    float s = 3.0e38f;
    if (f < n_feat) {
        const float* e = edges + static_cast<size_t>(f) * kGridEdgeStride;
        s = 0.f;
        for (int b = 0; b < 64; ++b) s += 1.f / fmaxf(e[(b + 1) << 6] - e[b << 6], 1e-7f);
    }
    score[f] = s;
}

__global__ void iota_kernel(int* __restrict__ v, int n) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) v[i] = i;
}

__global__ void grid_plan_kernel(const uint16_t* __restrict__ masks, int n_masks, long long N,
                                 const float* __restrict__ score, GridPlan* __restrict__ plans) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n_masks) return;
    GridPlan p;
    const uint32_t mask = masks[m];
    int d = 0;
    for (int j = 0; j < 15; ++j) {
        p.feat[j] = -1;
        if ((mask >> j) & 1u) p.feat[d++] = j;
    }
    for (int j = d; j < 15; ++j) p.feat[j] = -1;
    p.d = d;
    grid_bits_for(N, d, p.bits);
    const int c = d < kGridDims ? d : kGridDims;
    // the c features with the lowest concentration (ties: lower feature)
    uint32_t chosen = 0;
    for (int r = 0; r < c; ++r) {
        int best = -1;
        float bs = 0.f;
        for (int j = 0; j < d; ++j) {
            const int f = p.feat[j];
            if ((chosen >> f) & 1u) continue;
            const float s = score[f];
            if (best < 0 || s < bs) { best = f; bs = s; }
        }
        chosen |= 1u << best;
    }
    // grid dimensions in ascending feature order (the order of the distance chain: the cell lower
    // bounds of grid_join.cu rely on it), the unused leading dimensions empty
    int g = kGridDims - c;
    for (int u = 0; u < kGridDims - c; ++u) { p.idx_feat[u] = -1; p.idx_col[u] = 0; }
    for (int j = 0; j < d; ++j)
        if ((chosen >> p.feat[j]) & 1u) {
            p.idx_feat[g] = p.feat[j];
            p.idx_col[g] = j;
            ++g;
        }
    p.pad_ = 0;
    plans[m] = p;
}

__global__ void cell_keys_kernel(const uint16_t* __restrict__ bin12, int n_pad, int N,
                                 const GridPlan* __restrict__ plan, uint32_t* __restrict__ keys) {
    const GridPlan p = *plan;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
        uint32_t key = 0;
#pragma unroll
        for (int g = 0; g < kGridDims; ++g)
            if (p.bits[g] > 0) {
                const uint32_t b = bin12[static_cast<size_t>(p.idx_feat[g]) * n_pad + i] >> (kGridMasterBits - p.bits[g]);
                key = (key << p.bits[g]) | b;
            }
        keys[i] = key;
    }
}

// Compact rows in cell order, two objects interleaved: pair i holds sorted positions 2i and 2i+1,
// column j of the pair = (x[2i][feat j], x[2i+1][feat j]) -- the operand layout of the packed
// fp32 arithmetic of grid_join.cu.  Columns >= d and the partner of an odd last row are zero.
__global__ void gather_rows_kernel(const float* __restrict__ Xp, int N, const int* __restrict__ perm,
                                   const GridPlan* __restrict__ plan, int dp, float4* __restrict__ Xs) {
    const GridPlan p = *plan;
    const int g_per_pair = dp / 2;                       // float4 per pair: two columns x two objects
    const long long total = static_cast<long long>((N + 1) / 2) * g_per_pair;
    for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < total;
         i += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int pair = static_cast<int>(i / g_per_pair), g = static_cast<int>(i - static_cast<long long>(pair) * g_per_pair);
        const float* r0 = Xp + static_cast<size_t>(perm[2 * pair]) * kRowFloats;
        const float* r1 = 2 * pair + 1 < N ? Xp + static_cast<size_t>(perm[2 * pair + 1]) * kRowFloats : nullptr;
        float v[4];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int j = 2 * g + u;
            v[2 * u] = j < p.d ? r0[p.feat[j]] : 0.f;
            v[2 * u + 1] = (j < p.d && r1) ? r1[p.feat[j]] : 0.f;
        }
        Xs[i] = make_float4(v[0], v[1], v[2], v[3]);
    }
}

// cell_start[c] = first sorted position whose key is >= c; cell_start[n_cells] = N
__global__ void cell_start_kernel(const uint32_t* __restrict__ keys, int N, int n_cells, int* __restrict__ cell_start) {
    for (int pz = blockIdx.x * blockDim.x + threadIdx.x; pz <= N; pz += gridDim.x * blockDim.x) {
        const int prev = pz == 0 ? -1 : static_cast<int>(keys[pz - 1]);
        const int cur = pz == N ? n_cells : static_cast<int>(keys[pz]);
        for (int c = prev + 1; c <= cur; ++c) cell_start[c] = pz;
    }
}

__global__ void query_flags_kernel(const int* __restrict__ perm, int N, int q_begin, int q_end,
                                   unsigned char* __restrict__ flags) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
        const int id = perm[i];
        flags[i] = (id >= q_begin && id < q_end) ? 1 : 0;
    }
}

#ifndef GRID_ORDER_BIT
#define GRID_ORDER_BIT 22
#endif
// Work estimate of a join warp (32 consecutive queries of the sorted order): the largest squared distance
// from one of its queries to the object k sorted positions away -- what its threshold will be about after
// the seed window; the rows a warp walks and the candidates it scans grow with it.  A scheduling hint only.
__global__ void warp_cost_kernel(const float* __restrict__ Xs, const int* __restrict__ qlist, int nq, int N, int d,
                                 int dp, int k, uint32_t* __restrict__ cost) {
    const int g4 = dp / 2;                               // float4 per pair of objects
    const int n_warps = (nq + 31) / 32;
    const int lane = threadIdx.x & 31;
    for (int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; w < n_warps; w += (gridDim.x * blockDim.x) >> 5) {
        const int qi = w * 32 + lane;
        float c = 0.f;
        if (qi < nq) {
            const int pos = qlist ? qlist[qi] : qi;
            int other = pos + k < N ? pos + k : pos - k;
            if (other < 0) other = pos > 0 ? 0 : N - 1;
            const float* a = Xs + (static_cast<size_t>(pos >> 1) * g4) * 4 + (pos & 1);
            const float* b = Xs + (static_cast<size_t>(other >> 1) * g4) * 4 + (other & 1);
            for (int j = 0; j < d; ++j) {
                const int o = (j >> 1) * 4 + (j & 1) * 2;
                const float diff = a[o] - b[o];
                c += diff * diff;
            }
        }
        const uint32_t m = __reduce_max_sync(0xffffffffu, __float_as_uint(c));   // c >= 0: bit order = value order
        if (lane == 0) cost[w] = m;
    }
}

size_t cub_temp_bytes(int64_t N) {
    size_t a = 0, b = 0;
    const int n = static_cast<int>(N);
    cub::DeviceRadixSort::SortPairs(nullptr, a, static_cast<const uint32_t*>(nullptr), static_cast<uint32_t*>(nullptr),
                                    static_cast<const int*>(nullptr), static_cast<int*>(nullptr), n);
    cub::DeviceSelect::Flagged(nullptr, b, static_cast<const int*>(nullptr), static_cast<const unsigned char*>(nullptr),
                               static_cast<int*>(nullptr), static_cast<int*>(nullptr), n);
    return al(a > b ? a : b);
}

int n_pad_for(int64_t N) { return static_cast<int>((N + 31) / 32 * 32); }

}  // namespace

size_t grid_table_bytes(int64_t N) {
    const size_t n_pad = n_pad_for(N);
    return al(15 * kGridEdgeStride * 4) + al(15 * n_pad * 2) + 256 + al(n_pad * 4);
}

size_t grid_index_bytes(int64_t N) {
    const size_t n = static_cast<size_t>(N);
    return 3 * al(n * 4)                                   // keys_in, keys, perm
           + al((n / 16 + 16) * 4)                         // cell_start
           + al((n + kGridSlackRows) * 64)                 // compact rows (<= 16 floats)
           + al(n * 4) + al(n) + 256                       // qlist, flags, selected count
           + cub_temp_bytes(N);
}

void grid_index_carve(unsigned char* r, size_t bytes, int64_t N, GridIndex* ix) {
    const size_t n = static_cast<size_t>(N);
    ix->keys_in = reinterpret_cast<uint32_t*>(r); r += al(n * 4);
    ix->keys = reinterpret_cast<uint32_t*>(r); r += al(n * 4);
    ix->perm = reinterpret_cast<int*>(r); r += al(n * 4);
    ix->cell_start = reinterpret_cast<int*>(r); r += al((n / 16 + 16) * 4);
    ix->Xs = reinterpret_cast<float*>(r); r += al((n + kGridSlackRows) * 64);
    ix->qlist = reinterpret_cast<int*>(r); r += al(n * 4);
    r += al(n) + 256;                                      // flags + count sit right after qlist
    ix->cub_tmp = r;
    ix->cub_bytes = cub_temp_bytes(N);
    (void)bytes;
}

cudaError_t grid_table_build(const float* Xp, int N, int n_feat, GridTable* t, unsigned char* region,
                             unsigned char* index_region, size_t index_bytes, cudaStream_t st) {
    const int n_pad = n_pad_for(N);
    t->Xp = Xp;
    t->n_pad = n_pad;
    t->edges = reinterpret_cast<float*>(region); region += al(15 * kGridEdgeStride * 4);
    t->bin12 = reinterpret_cast<uint16_t*>(region); region += al(static_cast<size_t>(15) * n_pad * 2);
    t->score = reinterpret_cast<float*>(region); region += 256;
    t->iota = reinterpret_cast<int*>(region);
    GridIndex ix;
    grid_index_carve(index_region, index_bytes, N, &ix);   // scratch: the per-mask region is still free
    for (int f = 0; f < n_feat; ++f) {
        column_keys_kernel<<<kGrid, 256, 0, st>>>(Xp, N, f, ix.keys_in);
        cudaError_t e = cub::DeviceRadixSort::SortKeys(ix.cub_tmp, ix.cub_bytes, ix.keys_in, ix.keys, N, 0, 32, st);
        if (e != cudaSuccess) return e;
        float* edges = t->edges + static_cast<size_t>(f) * kGridEdgeStride;
        edges_kernel<<<(kGridMaster + 256) / 256, 256, 0, st>>>(ix.keys, N, edges);
        bins_kernel<<<kGrid, 256, 0, st>>>(Xp, N, f, edges, t->bin12 + static_cast<size_t>(f) * n_pad);
    }
    score_kernel<<<1, 32, 0, st>>>(t->edges, n_feat, t->score);
    iota_kernel<<<kGrid, 256, 0, st>>>(t->iota, n_pad);
    return cudaGetLastError();
}

cudaError_t grid_plan_launch(const uint16_t* d_masks, int n_masks, int64_t N, const GridTable& t,
                             GridPlan* d_plans, cudaStream_t st) {
    grid_plan_kernel<<<(n_masks + 127) / 128, 128, 0, st>>>(d_masks, n_masks, N, t.score, d_plans);
    return cudaGetLastError();
}

cudaError_t grid_index_build(const GridTable& t, const GridPlan* d_plan, int N, int d, const int bits[kGridDims],
                             int64_t q_begin, int64_t q_end, int knn_k, GridIndex* ix, cudaStream_t st) {
    const int total_bits = bits[0] + bits[1] + bits[2];
    const int n_cells = 1 << total_bits;
    const int dp = (d + 3) / 4 * 4;
    cell_keys_kernel<<<kGrid, 256, 0, st>>>(t.bin12, t.n_pad, N, d_plan, ix->keys_in);
    cudaError_t e = cub::DeviceRadixSort::SortPairs(ix->cub_tmp, ix->cub_bytes, ix->keys_in, ix->keys, t.iota, ix->perm,
                                                    N, 0, total_bits, st);
    if (e != cudaSuccess) return e;
    gather_rows_kernel<<<kGrid, 256, 0, st>>>(t.Xp, N, ix->perm, d_plan, dp, reinterpret_cast<float4*>(ix->Xs));
    cell_start_kernel<<<kGrid, 256, 0, st>>>(ix->keys, N, n_cells, ix->cell_start);
    if (q_begin > 0 || q_end < N) {
        unsigned char* flags = reinterpret_cast<unsigned char*>(ix->qlist) + al(static_cast<size_t>(N) * 4);
        int* n_sel = reinterpret_cast<int*>(flags + al(static_cast<size_t>(N)));
        query_flags_kernel<<<kGrid, 256, 0, st>>>(ix->perm, N, static_cast<int>(q_begin), static_cast<int>(q_end), flags);
        e = cub::DeviceSelect::Flagged(ix->cub_tmp, ix->cub_bytes, t.iota, flags, ix->qlist, n_sel, N, st);
        if (e != cudaSuccess) return e;
    }
    ix->warp_order = nullptr;
    if (knn_k > 0) {
        // heaviest warps first: the grid ends when its slowest warp does, and a heavy warp that starts late is
        // the tail (measured: SMs 15 % idle on average without this; join kernels of 64 masks of config 5 at
        // N = 10^6: 6.83 -> 5.56 s).  Not for the range joins: there either order costs 13 % -- neighbouring warps
        // scan the same runs, and taking them apart loses that locality while the work per warp is even anyway.
        // keys_in is free once the cells are sorted.
        const int nq = static_cast<int>(q_end - q_begin), n_warps = (nq + 31) / 32;
        uint32_t* cost = ix->keys_in;
        uint32_t* cost_sorted = cost + n_warps;
        int* order = reinterpret_cast<int*>(cost_sorted + n_warps);
        const bool sliced = q_begin > 0 || q_end < N;
        warp_cost_kernel<<<kGrid, 256, 0, st>>>(ix->Xs, sliced ? ix->qlist : nullptr, nq, N, d, dp, knn_k < N ? knn_k : N - 1, cost);
        e = cub::DeviceRadixSort::SortPairsDescending(ix->cub_tmp, ix->cub_bytes, cost, cost_sorted, t.iota, order, n_warps,
                                                      GRID_ORDER_BIT, 32, st);
        if (e != cudaSuccess) return e;
        ix->warp_order = order;
    }
    return cudaGetLastError();
}

}  // namespace snaps
