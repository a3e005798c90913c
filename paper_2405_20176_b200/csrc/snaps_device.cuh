// snaps_device.cuh -- device-side building blocks shared by the sub-lattice join kernels (sm_100a).
//
// Layouts of the staged table ("a1" in DESIGN.md).  Row-major copy Xp: row r of the caller's
// N x n_feat fp32 matrix becomes 20 floats (80 bytes): features 0..14, then 5 zeros; used for
// query rows, seed evaluations and as the gather source of the grid engine's compact rows.
// Blocked copy Xb (the candidate stream of the sub-lattice kernels): 32 rows per block, four
// feature groups of 32 float4 per block, read with four fully coalesced 128-bit loads per warp.
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
    int32_t pad_[2];
};
static_assert(sizeof(BatchDesc) % 16 == 0, "BatchDesc rows are read with 128-bit loads");

// Squared distance on a runtime mask between a staged row in global memory (80 bytes, 16-byte
// aligned: four 128-bit loads cover the 15 features) and a query row held in registers; features
// added in ascending order (slow paths only).
__device__ __forceinline__ float masked_d2(const float* __restrict__ row, const float (&q)[15], uint32_t mask) {
    const float4* r4 = reinterpret_cast<const float4*>(row);
    const float4 a0 = __ldg(r4), a1 = __ldg(r4 + 1), a2 = __ldg(r4 + 2), a3 = __ldg(r4 + 3);
    const float a[16] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w,
                         a2.x, a2.y, a2.z, a2.w, a3.x, a3.y, a3.z, a3.w};
    float acc = 0.f;
#pragma unroll
    for (int j = 0; j < 15; ++j) {
        float diff = a[j] - q[j];
        float sq = __fmul_rn(diff, diff);
        if ((mask >> j) & 1u) acc = __fadd_rn(acc, sq);
    }
    return acc;
}

// ---- the candidate stream and the group filter shared by knn_lattice.cu, range_lattice.cu and
// range_grid.cu (DESIGN.md 5.1 steps 1-2).

// One block of the blocked table in registers: lane = row 32t + lane.
struct Blk {
    float4 v0, v1, v2, v3;
};

__device__ __forceinline__ void load_block(Blk& dst, const float4* __restrict__ Xb, int t, int lane) {
    const float4* b = Xb + static_cast<size_t>(t) * 128 + lane;
    dst.v0 = __ldg(b);
    dst.v1 = __ldg(b + 32);
    dst.v2 = __ldg(b + 64);
    dst.v3 = __ldg(b + 96);
}

// Packed fp32 pairs (sm_100: add / mul / fma .rn.f32x2 -> SASS FADD2 / FMUL2 / FFMA2): two IEEE
// round-to-nearest results per issued instruction, bit-identical to the scalar operations.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

struct TrueTag { static constexpr bool value = true; };
struct FalseTag { static constexpr bool value = false; };

// The per-query, per-batch constants of the filter.
struct FilterQuery {
    f32x2 nq01, nq23, nq45;   // the query's lattice features, negated, in pairs: c - q = c + (-q)
    f32x2 w2[4], nwq2[4];     // high features 6..13 in pairs: diff = c*w - q*w with w in {0,1} (1 = feature in H)
    float w14, nwq14;         // high feature 14
};

__device__ __forceinline__ void filter_query_set_row(FilterQuery& f, const float (&qlo)[kLow]) {
    f.nq01 = pack2(-qlo[0], -qlo[1]);
    f.nq23 = pack2(-qlo[2], -qlo[3]);
    f.nq45 = pack2(-qlo[4], -qlo[5]);
}

__device__ __forceinline__ void filter_query_init(FilterQuery& f, const float (&qhi)[9], uint32_t H) {
    float w[9];
#pragma unroll
    for (int j = 0; j < 9; ++j) w[j] = ((H >> (kLow + j)) & 1u) ? 1.f : 0.f;
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        f.w2[p] = pack2(w[2 * p], w[2 * p + 1]);
        f.nwq2[p] = pack2(-(w[2 * p] * qhi[2 * p]), -(w[2 * p + 1] * qhi[2 * p + 1]));
    }
    f.w14 = w[8];
    f.nwq14 = -(w[8] * qhi[8]);
}

// What the refine step needs of a candidate that passed: the high-feature part of every sum and the
// six lattice squared differences.
struct PairTerms {
    float base;
    float sq[kLow];
};

// FILTER of one candidate (this lane's row of block r): the six lattice squared differences, the
// high-feature part `base`, the 16 partial sums X[u] over subsets u of features {2,3,4,5} (add-only),
// and the test of each X[u] -- a lower bound of the four sums X[u] (+sq0) (+sq1) of group u --
// against the group's largest threshold G[u].
// Arithmetic in packed pairs where two values take the same operation: the squared differences of
// features (0,1), (2,3), (4,5); base = two FMA chains over the even and the odd high features
// (6,8,10,12 and 7,9,11,13), their sum, then feature 14 -- one fixed order, used wherever a base is
// formed; the partial sums pairwise (X[2v], X[2v+1]) + (sq, sq).  45 scalar operations become 25.
// G0BOTH: group 0 = lattice slots {}, {0}, {1}, {0,1} and only {0,1} is asked for (the batch with
// H empty): its own sum is the group's bound -- X[0] alone would be 0 there and let every candidate through.
template <bool G0BOTH>
__device__ __forceinline__ bool lattice_filter(const Blk& r, const FilterQuery& f, const float (&G)[16],
                                               PairTerms& out) {
    // keep the padding word of the fourth load live until here: otherwise its register is handed
    // out as scratch while the prefetch is still in flight and the warp stalls on it
    asm volatile("" ::"f"(r.v3.w));
    const f32x2 d01 = add2(pack2(r.v0.x, r.v0.y), f.nq01);
    const f32x2 d23 = add2(pack2(r.v0.z, r.v0.w), f.nq23);
    const f32x2 d45 = add2(pack2(r.v1.x, r.v1.y), f.nq45);
    const f32x2 s01 = mul2(d01, d01), s23 = mul2(d23, d23), s45 = mul2(d45, d45);
    unpack2(s01, out.sq[0], out.sq[1]);
    unpack2(s23, out.sq[2], out.sq[3]);
    unpack2(s45, out.sq[4], out.sq[5]);
    f32x2 b2 = 0ull;
    {
        const f32x2 c67 = pack2(r.v1.z, r.v1.w), c89 = pack2(r.v2.x, r.v2.y), cab = pack2(r.v2.z, r.v2.w),
                    ccd = pack2(r.v3.x, r.v3.y);
        f32x2 d;
        d = fma2(c67, f.w2[0], f.nwq2[0]); b2 = fma2(d, d, b2);
        d = fma2(c89, f.w2[1], f.nwq2[1]); b2 = fma2(d, d, b2);
        d = fma2(cab, f.w2[2], f.nwq2[2]); b2 = fma2(d, d, b2);
        d = fma2(ccd, f.w2[3], f.nwq2[3]); b2 = fma2(d, d, b2);
    }
    float be, bo;
    unpack2(b2, be, bo);
    const float d14 = __fmaf_rn(r.v3.z, f.w14, f.nwq14);
    const float base = __fmaf_rn(d14, d14, __fadd_rn(be, bo));
    out.base = base;
    // X[u], u = subset of {2,3,4,5}: pairs (X[2v], X[2v+1]) = (., . + sq2)
    const f32x2 q3 = pack2(out.sq[3], out.sq[3]), q4 = pack2(out.sq[4], out.sq[4]), q5 = pack2(out.sq[5], out.sq[5]);
    f32x2 P[8];
    P[0] = pack2(base, __fadd_rn(base, out.sq[2]));
    P[1] = add2(P[0], q3);
    P[2] = add2(P[0], q4);
    P[3] = add2(P[1], q4);
#pragma unroll
    for (int v = 0; v < 4; ++v) P[4 + v] = add2(P[v], q5);
    float X[16];
#pragma unroll
    for (int v = 0; v < 8; ++v) unpack2(P[v], X[2 * v], X[2 * v + 1]);
    float x0 = X[0];
    if (G0BOTH) x0 = __fadd_rn(__fadd_rn(X[0], out.sq[0]), out.sq[1]);
    bool pa = x0 < G[0], pb = false;
#pragma unroll
    for (int u = 0; u < 16; u += 2) {
        if (u > 0) pa |= X[u] < G[u];
        pb |= X[u + 1] < G[u + 1];
    }
    return pa | pb;
}

// COMPACT: the lanes that passed append (id, base, sq0..5) to the warp's queue of 8-word entries,
// kept as two arrays of 128-bit halves (queue[slot], queue[queue_len + slot]) so that consecutive
// slots are 16 bytes apart: conflict-free 128-bit accesses.  Returns the number appended (warp-uniform).
__device__ __forceinline__ int queue_push(float4* queue, int queue_len, int qtail, bool pass, unsigned bal,
                                          unsigned lanes_below, int cand, const PairTerms& t) {
    if (pass) {
        float4* e = queue + (static_cast<unsigned>(qtail + __popc(bal & lanes_below)) % static_cast<unsigned>(queue_len));
        e[0] = make_float4(__int_as_float(cand), t.base, t.sq[0], t.sq[1]);
        e[queue_len] = make_float4(t.sq[2], t.sq[3], t.sq[4], t.sq[5]);
    }
    return __popc(bal);
}

// The 64 subset sums of a queued candidate in the fixed order (high features -> 2,3,4 -> 5 -> 0 -> 1),
// written as rows T = 0..31 of a 32 x 32 transpose (row stride 36 words), half = 0: the sums without
// feature 5, half = 1: with it.  X8 = partial sums over features 2,3,4.
__device__ __forceinline__ void lattice_partial8(const PairTerms& t, float (&X8)[8]) {
    X8[0] = t.base;
#pragma unroll
    for (int u = 1; u < 8; ++u) {
        const int hb = 31 - __clz(u);
        X8[u] = __fadd_rn(X8[u & ~(1 << hb)], t.sq[2 + hb]);
    }
}

// The four sums of group 4*uu (+ 32*half) in that order: lattice subsets T = 4*uu + {0, 1, 2, 3}.
__device__ __forceinline__ void lattice_group_sums(const PairTerms& t, const float (&X8)[8], int half, int uu,
                                                   float& s0, float& s1, float& s2, float& s3) {
    s0 = half ? __fadd_rn(X8[uu], t.sq[5]) : X8[uu];
    s1 = __fadd_rn(s0, t.sq[0]);
    s2 = __fadd_rn(s0, t.sq[1]);
    s3 = __fadd_rn(s1, t.sq[1]);
}

__device__ __forceinline__ void lattice_sums_to_transpose(const PairTerms& t, const float (&X8)[8], int half,
                                                          float* mt, int lane) {
#pragma unroll
    for (int uu = 0; uu < 8; ++uu) {
        float s0, s1, s2, s3;
        lattice_group_sums(t, X8, half, uu, s0, s1, s2, s3);
        mt[(4 * uu + 0) * 36 + lane] = s0;
        mt[(4 * uu + 1) * 36 + lane] = s1;
        mt[(4 * uu + 2) * 36 + lane] = s2;
        mt[(4 * uu + 3) * 36 + lane] = s3;
    }
}

// Whether any of a candidate's 64 sums is below its list's threshold (thr[T], T = 0..63, read as
// 128-bit broadcasts): the same values, formed in the same order, as the refine step compares.
__device__ __forceinline__ bool lattice_any_below(const PairTerms& t, const float (&X8)[8], const float* thr) {
    bool pass = false;
#pragma unroll
    for (int half = 0; half < 2; ++half) {
#pragma unroll
        for (int uu = 0; uu < 8; ++uu) {
            float s0, s1, s2, s3;
            lattice_group_sums(t, X8, half, uu, s0, s1, s2, s3);
            const float4 h = *reinterpret_cast<const float4*>(thr + 32 * half + 4 * uu);
            pass |= (s0 < h.x) | (s1 < h.y) | (s2 < h.z) | (s3 < h.w);
        }
    }
    return pass;
}

// The entry a lane takes from the queue at refine time; self (reading A4) and padding rows (A19)
// get an infinite base so that none of their sums can pass.
__device__ __forceinline__ int queue_pop(const float4* queue, int queue_len, int head, int lane, int n, int q, int N,
                                         PairTerms& t) {
    t.base = __int_as_float(0x7f800000);
#pragma unroll
    for (int j = 0; j < kLow; ++j) t.sq[j] = 0.f;
    int cand = -1;
    if (lane < n) {
        const float4* e = queue + (static_cast<unsigned>(head + lane) % static_cast<unsigned>(queue_len));
        const float4 a = e[0], b = e[queue_len];
        cand = __float_as_int(a.x);
        t.base = a.y; t.sq[0] = a.z; t.sq[1] = a.w;
        t.sq[2] = b.x; t.sq[3] = b.y; t.sq[4] = b.z; t.sq[5] = b.w;
        if (cand == q || cand >= N) t.base = __int_as_float(0x7f800000);
    }
    return cand;
}

// EXACT TEST (between COMPACT and REFINE): the group filter lets a candidate through when a lower
// bound of four sums is below the largest of four thresholds; most of those candidates enter no
// list.  Lanes 0..n-1 take the n oldest queue entries (lane = candidate), form the 64 sums exactly
// as the refine step does and compare each with its list's current threshold thr[T] (16 broadcast
// reads); only candidates with a sum below a threshold go on, in order, to the survivors' array
// surv (32 entries as two arrays of 128-bit halves; nb of them already wait), and the refine step
// -- whose cost does not depend on how many of its 32 candidates count -- runs when 32 of them
// wait.  Thresholds never rise, so a candidate dropped here could not count later.  When the array
// fills up, the entries behind the last survivor taken stay queued and are tested again after the
// refine step.  Returns (entries consumed) | (survivors now waiting) << 8.
__device__ __forceinline__ int lattice_exact_test(const float4* queue, int queue_len, float4* surv, const float* thr,
                                                  int lane, int q, int N, int head, int n, int nb) {
    PairTerms pt;
    const int cand = queue_pop(queue, queue_len, head, lane, n, q, N, pt);
    float X8[8];
    lattice_partial8(pt, X8);
    const bool pass = lattice_any_below(pt, X8, thr);
    const unsigned sb = __ballot_sync(kFull, pass);
    const int pos = nb + __popc(sb & ((1u << lane) - 1u));
    const bool take = pass && pos < 32;
    if (take) {
        surv[pos] = make_float4(__int_as_float(cand), pt.base, pt.sq[0], pt.sq[1]);
        surv[32 + pos] = make_float4(pt.sq[2], pt.sq[3], pt.sq[4], pt.sq[5]);
    }
    const int tot = nb + __popc(sb);
    if (tot <= 32) return n | (tot << 8);
    const unsigned last = __ballot_sync(kFull, take && pos == 31);
    return __ffs(last) | (32 << 8);
}

// The survivor a lane takes at refine time (lanes >= n: an infinite base, no sum can pass).
__device__ __forceinline__ int survivors_pop(const float4* surv, int lane, int n, PairTerms& t) {
    t.base = __int_as_float(0x7f800000);
#pragma unroll
    for (int j = 0; j < kLow; ++j) t.sq[j] = 0.f;
    int cand = -1;
    if (lane < n) {
        const float4 a = surv[lane], b = surv[32 + lane];
        cand = __float_as_int(a.x);
        t.base = a.y; t.sq[0] = a.z; t.sq[1] = a.w;
        t.sq[2] = b.x; t.sq[3] = b.y; t.sq[4] = b.z; t.sq[5] = b.w;
    }
    return cand;
}

}  // namespace snaps
