// eps_search.cu -- NEXT-2: the search radius for a target selectivity from a
// sampled distance histogram.  "The distances between a sample of points and points within the
// dataset are computed to create a histogram of distances between points.  Using this histogram,
// a cumulative distance distribution histogram is computed which yields the relationship between
// a search distance and the average number of neighbors" -- selectivity s = mean neighbours per
// point, self excluded.  Device: the histogram of D(q, c; mask) over sampled
// queries x sampled candidates (q != c) per mask.  Host: cumulative histogram -> radius.
#include "eps_search.cuh"

namespace snaps {

__global__ void gather_rows_kernel(const float* __restrict__ X, int64_t ld, int n_feat,
                                   const int32_t* __restrict__ ids, int n, float* __restrict__ out) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n * 16; i += gridDim.x * blockDim.x) {
        const int r = i >> 4, j = i & 15;
        out[i] = j < n_feat ? X[static_cast<int64_t>(ids[r]) * ld + j] : 0.f;
    }
}

// grid = (n_masks, query chunks); one thread per (query of the chunk) loops over all candidates
__global__ void dist_hist_kernel(const float* __restrict__ Xq, const int32_t* __restrict__ qid, int nq,
                                 const float* __restrict__ Xc, const int32_t* __restrict__ cid, int nc,
                                 const uint16_t* __restrict__ masks, const float* __restrict__ rmax, int n_bins,
                                 unsigned long long* __restrict__ hist) {
    extern __shared__ unsigned int sh[];
    const int m = blockIdx.x;
    for (int i = threadIdx.x; i < n_bins; i += blockDim.x) sh[i] = 0u;
    __syncthreads();
    const uint32_t mask = masks[m];
    const float scale = static_cast<float>(n_bins) / rmax[m];
    for (int qi = blockIdx.y * blockDim.x + threadIdx.x; qi < nq; qi += gridDim.y * blockDim.x) {
        float q[15];
#pragma unroll
        for (int j = 0; j < 15; ++j) q[j] = Xq[qi * 16 + j];
        const int my = qid[qi];
        for (int ci = 0; ci < nc; ++ci) {
            if (cid[ci] == my) continue;   // self excluded by index
            const float* c = Xc + ci * 16;
            float acc = 0.f;
#pragma unroll
            for (int j = 0; j < 15; ++j) {
                const float diff = c[j] - q[j];
                const float sq = __fmul_rn(diff, diff);
                if ((mask >> j) & 1u) acc = __fadd_rn(acc, sq);
            }
            const float b = sqrtf(acc) * scale;
            if (b < static_cast<float>(n_bins)) atomicAdd(&sh[static_cast<int>(b)], 1u);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n_bins; i += blockDim.x)
        if (sh[i]) atomicAdd(&hist[static_cast<size_t>(m) * n_bins + i], static_cast<unsigned long long>(sh[i]));
}

// eps_mean ("it samples the dataset to first estimate the mean distance between points
// in a dataset (eps_mean), which is used as the upper bound on a practical search radius"): the mean of
// D over the sampled (query, candidate) pairs, c != q by index.  One block per (mask, query chunk)
// writes its partial sum; mean_finish_kernel adds the partials in a fixed order (deterministic).
__global__ void mean_dist_kernel(const float* __restrict__ Xq, const int32_t* __restrict__ qid, int nq,
                                 const float* __restrict__ Xc, const int32_t* __restrict__ cid, int nc,
                                 const uint16_t* __restrict__ masks, double* __restrict__ partial) {
    __shared__ double red[128];
    const int m = blockIdx.x;
    const uint32_t mask = masks[m];
    double tot = 0.0;
    for (int qi = blockIdx.y * blockDim.x + threadIdx.x; qi < nq; qi += gridDim.y * blockDim.x) {
        float q[15];
#pragma unroll
        for (int j = 0; j < 15; ++j) q[j] = Xq[qi * 16 + j];
        const int my = qid[qi];
        for (int c0 = 0; c0 < nc; c0 += 256) {
            float part = 0.f;                       // fp32 over 256 candidates, fp64 across chunks
            const int c1 = min(nc, c0 + 256);
            for (int ci = c0; ci < c1; ++ci) {
                if (cid[ci] == my) continue;
                const float* c = Xc + ci * 16;
                float acc = 0.f;
#pragma unroll
                for (int j = 0; j < 15; ++j) {
                    const float diff = c[j] - q[j];
                    const float sq = __fmul_rn(diff, diff);
                    if ((mask >> j) & 1u) acc = __fadd_rn(acc, sq);
                }
                part += sqrtf(acc);
            }
            tot += static_cast<double>(part);
        }
    }
    red[threadIdx.x] = tot;
    __syncthreads();
    for (int s = 64; s > 0; s >>= 1) {
        if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[static_cast<size_t>(m) * gridDim.y + blockIdx.y] = red[0];
}

__global__ void mean_finish_kernel(const double* __restrict__ partial, int chunks, int n_masks, double pairs,
                                   float* __restrict__ eps_mean) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n_masks) return;
    double s = 0.0;
    for (int c = 0; c < chunks; ++c) s += partial[static_cast<size_t>(m) * chunks + c];
    eps_mean[m] = static_cast<float>(s / pairs);
}

// Cumulative histogram -> radii: for every target selectivity the upper edge of the first bin whose
// cumulative mean neighbour count cum * (N-1) / pairs reaches it; eps_mean (the histogram's range) if none does.
__global__ void eps_from_hist_kernel(const unsigned long long* __restrict__ hist, int n_masks, int n_bins,
                                     const float* __restrict__ rmax, double N_minus_1, double pairs,
                                     const double* __restrict__ targets, int n_targets, float* __restrict__ eps) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_masks * n_targets) return;
    const int m = i / n_targets, t = i - m * n_targets;
    const double target = targets[t];
    unsigned long long cum = 0;
    float e = rmax[m];
    for (int b = 0; b < n_bins; ++b) {
        cum += hist[static_cast<size_t>(m) * n_bins + b];
        if (static_cast<double>(cum) * N_minus_1 / pairs >= target) {
            e = static_cast<float>(static_cast<double>(rmax[m]) * (b + 1) / n_bins);
            break;
        }
    }
    eps[i] = e;
}

// The eps grid G (Fig. 3 "evenly spaced search distances"): G radii from eps_min to eps_max in
// fp32, eps_g = eps_min + g * ((eps_max - eps_min) / (G - 1)) with every operation rounded, the last one
// eps_max itself; beside it the squared thresholds the join kernels compare with (closed ball, reading A2:
// fl(eps^2) for the grid engine, its successor for the sub-lattice engine's strict compare).
__global__ void eps_grid_kernel(const float* __restrict__ eps_mm, int n_masks, int G, int successor,
                                float* __restrict__ eps_grid, float* __restrict__ thr) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_masks * G) return;
    const int m = i / G, g = i - m * G;
    const float e_min = eps_mm[2 * m], e_max = eps_mm[2 * m + 1];
    const float step = __fdiv_rn(__fsub_rn(e_max, e_min), static_cast<float>(G - 1));
    const float e = g == G - 1 ? e_max : __fadd_rn(e_min, __fmul_rn(static_cast<float>(g), step));
    const float e2 = static_cast<float>(static_cast<double>(e) * static_cast<double>(e));
    eps_grid[i] = e;
    thr[i] = successor ? nextafterf(e2, __int_as_float(0x7f800000)) : e2;
}

cudaError_t eps_grid_launch(const float* eps_mm, int n_masks, int G, int successor, float* eps_grid, float* thr,
                            cudaStream_t st) {
    eps_grid_kernel<<<(n_masks * G + 127) / 128, 128, 0, st>>>(eps_mm, n_masks, G, successor, eps_grid, thr);
    return cudaGetLastError();
}

size_t dist_hist_workspace_bytes(int nq, int nc, int n_masks) {
    auto al = [](size_t x) { return (x + 255) / 256 * 256; };
    return al(static_cast<size_t>(nq) * 64) + al(static_cast<size_t>(nc) * 64) + al(static_cast<size_t>(nq) * 4) +
           al(static_cast<size_t>(nc) * 4) + al(static_cast<size_t>(n_masks) * 2) + al(static_cast<size_t>(n_masks) * 4);
}

size_t eps_search_workspace_bytes(int nq, int nc, int n_masks, int n_bins, int n_targets) {
    auto al = [](size_t x) { return (x + 255) / 256 * 256; };
    return dist_hist_workspace_bytes(nq, nc, n_masks) + al(static_cast<size_t>(n_masks) * 16 * 8) +
           al(static_cast<size_t>(n_masks) * n_bins * 8) + al(static_cast<size_t>(n_targets) * 8);
}

cudaError_t dist_hist_launch(const float* X, int64_t ld, int n_feat, const int32_t* h_q, int nq, const int32_t* h_c,
                             int nc, const uint16_t* h_masks, const float* h_rmax, int n_masks, int n_bins,
                             unsigned long long* out_hist, void* ws, cudaStream_t st) {
    auto al = [](size_t x) { return (x + 255) / 256 * 256; };
    unsigned char* p = static_cast<unsigned char*>(ws);
    float* Xq = reinterpret_cast<float*>(p); p += al(static_cast<size_t>(nq) * 64);
    float* Xc = reinterpret_cast<float*>(p); p += al(static_cast<size_t>(nc) * 64);
    int32_t* dq = reinterpret_cast<int32_t*>(p); p += al(static_cast<size_t>(nq) * 4);
    int32_t* dc = reinterpret_cast<int32_t*>(p); p += al(static_cast<size_t>(nc) * 4);
    uint16_t* dm = reinterpret_cast<uint16_t*>(p); p += al(static_cast<size_t>(n_masks) * 2);
    float* dr = reinterpret_cast<float*>(p);
    cudaError_t e;
    if ((e = cudaMemcpyAsync(dq, h_q, sizeof(int32_t) * nq, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(dc, h_c, sizeof(int32_t) * nc, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(dm, h_masks, sizeof(uint16_t) * n_masks, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(dr, h_rmax, sizeof(float) * n_masks, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(out_hist, 0, sizeof(unsigned long long) * static_cast<size_t>(n_masks) * n_bins, st)) != cudaSuccess) return e;
    gather_rows_kernel<<<(nq * 16 + 255) / 256, 256, 0, st>>>(X, ld, n_feat, dq, nq, Xq);
    gather_rows_kernel<<<(nc * 16 + 255) / 256, 256, 0, st>>>(X, ld, n_feat, dc, nc, Xc);
    const int chunks = (nq + 127) / 128 < 16 ? (nq + 127) / 128 : 16;
    dist_hist_kernel<<<dim3(n_masks, chunks), 128, static_cast<size_t>(n_bins) * 4, st>>>(Xq, dq, nq, Xc, dc, nc, dm, dr,
                                                                                         n_bins, out_hist);
    return cudaGetLastError();
}

cudaError_t eps_search_launch(const float* X, int64_t N, int64_t ld, int n_feat, const int32_t* h_q, int nq, const int32_t* h_c,
                              int nc, long long pairs, const uint16_t* h_masks, int n_masks, int n_bins,
                              const double* h_targets, int n_targets, float* out_eps_mean, float* out_eps,
                              unsigned long long* out_hist, void* ws, cudaStream_t st) {
    auto al = [](size_t x) { return (x + 255) / 256 * 256; };
    unsigned char* p = static_cast<unsigned char*>(ws);
    float* Xq = reinterpret_cast<float*>(p); p += al(static_cast<size_t>(nq) * 64);
    float* Xc = reinterpret_cast<float*>(p); p += al(static_cast<size_t>(nc) * 64);
    int32_t* dq = reinterpret_cast<int32_t*>(p); p += al(static_cast<size_t>(nq) * 4);
    int32_t* dc = reinterpret_cast<int32_t*>(p); p += al(static_cast<size_t>(nc) * 4);
    uint16_t* dm = reinterpret_cast<uint16_t*>(p); p += al(static_cast<size_t>(n_masks) * 2);
    p += al(static_cast<size_t>(n_masks) * 4);
    double* partial = reinterpret_cast<double*>(p); p += al(static_cast<size_t>(n_masks) * 16 * 8);
    unsigned long long* hist_ws = reinterpret_cast<unsigned long long*>(p); p += al(static_cast<size_t>(n_masks) * n_bins * 8);
    double* d_targets = reinterpret_cast<double*>(p);
    unsigned long long* hist = out_hist ? out_hist : hist_ws;
    cudaError_t e;
    if ((e = cudaMemcpyAsync(dq, h_q, sizeof(int32_t) * nq, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(dc, h_c, sizeof(int32_t) * nc, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(dm, h_masks, sizeof(uint16_t) * n_masks, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(d_targets, h_targets, sizeof(double) * n_targets, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(hist, 0, sizeof(unsigned long long) * static_cast<size_t>(n_masks) * n_bins, st)) != cudaSuccess) return e;
    gather_rows_kernel<<<(nq * 16 + 255) / 256, 256, 0, st>>>(X, ld, n_feat, dq, nq, Xq);
    gather_rows_kernel<<<(nc * 16 + 255) / 256, 256, 0, st>>>(X, ld, n_feat, dc, nc, Xc);
    const int chunks = (nq + 127) / 128 < 16 ? (nq + 127) / 128 : 16;
    mean_dist_kernel<<<dim3(n_masks, chunks), 128, 0, st>>>(Xq, dq, nq, Xc, dc, nc, dm, partial);
    mean_finish_kernel<<<(n_masks + 127) / 128, 128, 0, st>>>(partial, chunks, n_masks, static_cast<double>(pairs), out_eps_mean);
    dist_hist_kernel<<<dim3(n_masks, chunks), 128, static_cast<size_t>(n_bins) * 4, st>>>(Xq, dq, nq, Xc, dc, nc, dm, out_eps_mean,
                                                                                         n_bins, hist);
    eps_from_hist_kernel<<<(n_masks * n_targets + 127) / 128, 128, 0, st>>>(hist, n_masks, n_bins, out_eps_mean,
                                                                            static_cast<double>(N - 1), static_cast<double>(pairs),
                                                                            d_targets, n_targets, out_eps);
    return cudaGetLastError();
}

}  // namespace snaps
