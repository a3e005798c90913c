/*
 * snaps_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 brute-force CPU statement of what the SNAPS hot path
 * computes (arXiv 2405.20176; line numbers are /root/reference/PAPER.md).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.  It shares no code, header,
 * table or helper with the CUDA path under paper_2405_20176_b200/.
 *
 * Both joins have a plain definition that any index or reuse scheme reaches
 * exactly, so the oracle IS that definition:
 *
 *   D2(i,j;S) = sum_{f in S} (X[i,f] - X[j,f])^2, fp64, f increasing
 *   D(i,j;S)  = sqrt(D2)                    Euclidean: DESIGN.md reading A1
 *
 *   kNNSJ: for every query i the k objects j != i with
 *       the smallest key (D2, j); self excluded BY INDEX (PAPER.md:221,
 *       reading A4), ties to the smaller id (reading A3).
 *   DSSJ: cnt[i] = #{j != i : D(i,j) <= eps}  (closed
 *       ball, reading A2), sum[i] = sum of those D.
 *   Scores: kth = D_(k); mean = (1/k) sum D_(r)
 *       (mean of distances, reading A5); indeg[j] = #{i : j in kNN(i)};
 *       epsmean = sum/cnt, 0 when cnt == 0 (reading A6).
 *
 * Selection is k passes of "smallest not yet taken key (D2, j)" over the
 * full distance row -- a truncated selection sort, no heap, no pruning, no
 * sharing of work between masks or queries.
 *
 * Pins (tests/test_oracle_*.py): Eq. 1 mask count; one-feature and
 * duplicated-column closed forms; 1-D lattice closed form; {0,1}^d hypercube
 * closed-form counts and order statistics; scipy cKDTree on random tables;
 * exhaustive k-subset enumeration for N <= 8; invariants of PAPER.md:136,
 * 221, 235.  Table 2's metric VALUES are "parity unpinned" (Figure 1's
 * coordinates are not in the text); only its internal sums are checked.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_BAD_ARG 1
#define ORACLE_NO_MEM 2

int snaps_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* D2(i, j; S), fp64, features in increasing order (definition 1 above). */
static double dist2(const float *X, int64_t ld, int n_feat, uint16_t S,
                    int64_t i, int64_t j)
{
    double acc = 0.0;
    for (int f = 0; f < n_feat; ++f) {
        if ((S >> f) & 1u) {
            double diff = (double)X[i * ld + f] - (double)X[j * ld + f];
            acc += diff * diff;
        }
    }
    return acc;
}

static int check_common(const float *X, int64_t N, int n_feat, int64_t ld,
                        const uint16_t *masks, int n_masks)
{
    if (!X || !masks || N < 2 || n_feat < 1 || n_feat > 15 || ld < n_feat || n_masks < 1)
        return ORACLE_BAD_ARG;
    for (int m = 0; m < n_masks; ++m)
        if (masks[m] == 0 || (masks[m] >> n_feat) != 0)
            return ORACLE_BAD_ARG;
    return ORACLE_OK;
}

/*
 * kNN self-join.  qids == NULL means queries 0..N-1 (then nq must be N).
 * out_idx, out_dist: [n_masks][nq][k]; out_dist holds D (not D2), ascending.
 */
int snaps_oracle_knn(const float *X, int64_t N, int n_feat, int64_t ld,
                     const uint16_t *masks, int n_masks, int k,
                     const int64_t *qids, int64_t nq,
                     int32_t *out_idx, double *out_dist)
{
    int rc = check_common(X, N, n_feat, ld, masks, n_masks);
    if (rc) return rc;
    if (k < 1 || k > N - 1 || nq < 1 || !out_idx || !out_dist) return ORACLE_BAD_ARG;
    if (!qids && nq != N) return ORACLE_BAD_ARG;
    int failed = 0;
#pragma omp parallel
    {
        double *row = (double *)malloc((size_t)N * sizeof(double));
        char *taken = (char *)malloc((size_t)N);
        if (!row || !taken) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp barrier
        if (!failed) {
#pragma omp for collapse(2) schedule(dynamic, 4)
            for (int m = 0; m < n_masks; ++m) {
                for (int64_t q = 0; q < nq; ++q) {
                    int64_t i = qids ? qids[q] : q;
                    uint16_t S = masks[m];
                    for (int64_t j = 0; j < N; ++j) row[j] = dist2(X, ld, n_feat, S, i, j);
                    memset(taken, 0, (size_t)N);
                    taken[i] = 1; /* self excluded by index */
                    for (int r = 0; r < k; ++r) {
                        int64_t best = -1;
                        for (int64_t j = 0; j < N; ++j) {
                            /* strict '<' while scanning j upward = key (D2, j) */
                            if (!taken[j] && (best < 0 || row[j] < row[best])) best = j;
                        }
                        taken[best] = 1;
                        size_t o = ((size_t)m * (size_t)nq + (size_t)q) * (size_t)k + (size_t)r;
                        out_idx[o] = (int32_t)best;
                        out_dist[o] = sqrt(row[best]);
                    }
                }
            }
        }
        free(row);
        free(taken);
    }
    return failed ? ORACLE_NO_MEM : ORACLE_OK;
}

/*
 * kNN scores from full lists (all N queries).  idx/dist: [n_masks][N][k].
 * out_kth, out_mean: [n_masks][N] fp64; out_indeg: [n_masks][N] int64.
 */
int snaps_oracle_knn_scores(int64_t N, int n_masks, int k,
                            const int32_t *idx, const double *dist,
                            double *out_kth, double *out_mean, int64_t *out_indeg)
{
    if (N < 2 || n_masks < 1 || k < 1 || !idx || !dist) return ORACLE_BAD_ARG;
    for (int m = 0; m < n_masks; ++m) {
        if (out_indeg)
            for (int64_t j = 0; j < N; ++j) out_indeg[(size_t)m * N + j] = 0;
        for (int64_t i = 0; i < N; ++i) {
            size_t o = ((size_t)m * N + i) * (size_t)k;
            double s = 0.0;
            for (int r = 0; r < k; ++r) {
                s += dist[o + r];
                if (out_indeg) {
                    int32_t j = idx[o + r];
                    if (j < 0 || j >= N) return ORACLE_BAD_ARG;
                    out_indeg[(size_t)m * N + j] += 1;
                }
            }
            if (out_kth) out_kth[(size_t)m * N + i] = dist[o + k - 1];
            if (out_mean) out_mean[(size_t)m * N + i] = s / (double)k;
        }
    }
    return ORACLE_OK;
}

/*
 * eps range self-join.  eps: [n_masks] fp64.  out_cnt: [n_masks][nq] int64,
 * out_sum: [n_masks][nq] fp64 (sum of D over the counted neighbours),
 * out_mean: [n_masks][nq] fp64 = sum/cnt or 0 (any output may be NULL).
 */
int snaps_oracle_range(const float *X, int64_t N, int n_feat, int64_t ld,
                       const uint16_t *masks, int n_masks, const double *eps,
                       const int64_t *qids, int64_t nq,
                       int64_t *out_cnt, double *out_sum, double *out_mean)
{
    int rc = check_common(X, N, n_feat, ld, masks, n_masks);
    if (rc) return rc;
    if (!eps || nq < 1) return ORACLE_BAD_ARG;
    if (!qids && nq != N) return ORACLE_BAD_ARG;
    for (int m = 0; m < n_masks; ++m)
        if (!(eps[m] > 0.0) || !isfinite(eps[m])) return ORACLE_BAD_ARG;
#pragma omp parallel for collapse(2) schedule(dynamic, 16)
    for (int m = 0; m < n_masks; ++m) {
        for (int64_t q = 0; q < nq; ++q) {
            int64_t i = qids ? qids[q] : q;
            int64_t c = 0;
            double s = 0.0;
            for (int64_t j = 0; j < N; ++j) {
                if (j == i) continue;
                double D = sqrt(dist2(X, ld, n_feat, masks[m], i, j));
                if (D <= eps[m]) {
                    c += 1;
                    s += D;
                }
            }
            size_t o = (size_t)m * (size_t)nq + (size_t)q;
            if (out_cnt) out_cnt[o] = c;
            if (out_sum) out_sum[o] = s;
            if (out_mean) out_mean[o] = (c > 0) ? s / (double)c : 0.0;
        }
    }
    return ORACLE_OK;
}

/* All D(i, j; S) for one query row, fp64: used by tests that need the raw row
 * (gap rule of reading A3, the 1e-6 band of reading A2). out: [N], out[i] = 0. */
int snaps_oracle_dist_row(const float *X, int64_t N, int n_feat, int64_t ld,
                          uint16_t mask, int64_t i, double *out)
{
    if (!X || !out || N < 1 || n_feat < 1 || n_feat > 15 || ld < n_feat || i < 0 || i >= N)
        return ORACLE_BAD_ARG;
    for (int64_t j = 0; j < N; ++j) out[j] = sqrt(dist2(X, ld, n_feat, mask, i, j));
    return ORACLE_OK;
}
