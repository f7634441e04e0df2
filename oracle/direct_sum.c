/* O6 in plain C — ORACLE CODE (test infrastructure; also the timed CPU baseline).
 *
 *   p(x) = 2^{-K} * sum_{k in {I,X,Y,Z}^K} prod_{s=1..m} T_s[ idx_s(k), x_s ]
 *
 * Eq. 1 of the paper with the 1/2-per-cut constant (reading
 * G1).  This is the "prior method" the paper improves on: all 4^|E| cut-basis
 * assignments are enumerated.  The enumeration is a depth-first
 * odometer over the cuts e = 0..K-1 that carries the running product of the subcircuits
 * whose last incident cut has already been assigned — still the literal sum, every one of
 * the 4^K terms is visited, in float64.  Parallel over states (OpenMP), nothing else.
 *
 * Shares no code with the CUDA library.
 */
#include <stdint.h>
#include <stdlib.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int K, m;
    /* for each cut e: the subcircuits incident on it and the stride of e's digit in their row index */
    const int *inc_sub;      /* [K][2] */
    const int64_t *inc_str;  /* [K][2] */
    /* subcircuits whose LAST incident cut is e: closes[close_ofs[e] .. close_ofs[e+1]) */
    const int *close_ofs;    /* [K+1] */
    const int *closes;
    const double *const *col; /* col[s] = pointer to the x_s slice, element i at col[s][i*stride_s] */
    const int64_t *col_stride; /* [m] = 2^{o_s} */
} ctx_t;

static double rec(const ctx_t *c, int e, int64_t *idx, double partial)
{
    if (e == c->K) return partial;
    const int s0 = c->inc_sub[2 * e], s1 = c->inc_sub[2 * e + 1];
    const int64_t st0 = c->inc_str[2 * e], st1 = c->inc_str[2 * e + 1];
    double acc = 0.0;
    for (int k = 0; k < 4; ++k) {
        idx[s0] += k * st0;
        idx[s1] += k * st1;
        double p = partial;
        for (int j = c->close_ofs[e]; j < c->close_ofs[e + 1]; ++j) {
            const int s = c->closes[j];
            p *= c->col[s][idx[s] * c->col_stride[s]];
        }
        acc += rec(c, e + 1, idx, p);
        idx[s0] -= k * st0;
        idx[s1] -= k * st1;
    }
    return acc;
}

/* tensors[s]: [4^{c_s}][2^{o_s}] row-major float64.  keys: [B][m] int64 (x_s per state).
 * sub_cuts: concatenated incident-cut lists (axis order, first = most significant), offsets in sub_ofs[m+1].
 * Returns the number of threads used. */
int tqc_oracle_direct_sum(int m, int K, const int *sub_ofs, const int *sub_cuts,
                          const double *const *tensors, const int64_t *two_pow_o,
                          const int64_t *keys, int64_t B, double *out, int num_threads)
{
    int *inc_sub = (int *)malloc(sizeof(int) * 2 * (K > 0 ? K : 1));
    int64_t *inc_str = (int64_t *)malloc(sizeof(int64_t) * 2 * (K > 0 ? K : 1));
    int *fill = (int *)calloc(K > 0 ? K : 1, sizeof(int));
    int *last = (int *)malloc(sizeof(int) * m);
    for (int s = 0; s < m; ++s) {
        int c = sub_ofs[s + 1] - sub_ofs[s];
        last[s] = -1;
        for (int j = 0; j < c; ++j) {
            int e = sub_cuts[sub_ofs[s] + j];
            int64_t stride = 1;
            for (int t = j + 1; t < c; ++t) stride *= 4;
            inc_sub[2 * e + fill[e]] = s;
            inc_str[2 * e + fill[e]] = stride;
            fill[e]++;
            if (e > last[s]) last[s] = e;
        }
    }
    int *close_ofs = (int *)calloc(K + 2, sizeof(int));
    int *closes = (int *)malloc(sizeof(int) * (m > 0 ? m : 1));
    for (int s = 0; s < m; ++s) if (last[s] >= 0) close_ofs[last[s] + 1]++;
    for (int e = 0; e < K; ++e) close_ofs[e + 1] += close_ofs[e];
    int *pos = (int *)malloc(sizeof(int) * (K + 1));
    for (int e = 0; e <= K; ++e) pos[e] = close_ofs[e];
    for (int s = 0; s < m; ++s) if (last[s] >= 0) closes[pos[last[s]]++] = s;

    int used = 1;
#ifdef _OPENMP
    if (num_threads > 0) omp_set_num_threads(num_threads);
    used = omp_get_max_threads();
#endif
    const double scale = ldexp(1.0, -K);
#pragma omp parallel
    {
        int64_t *idx = (int64_t *)calloc(m > 0 ? m : 1, sizeof(int64_t));
        const double **col = (const double **)malloc(sizeof(double *) * (m > 0 ? m : 1));
        ctx_t c = {K, m, inc_sub, inc_str, close_ofs, closes, col, two_pow_o};
#pragma omp for schedule(dynamic, 1)
        for (int64_t b = 0; b < B; ++b) {
            double pre = 1.0;
            for (int s = 0; s < m; ++s) {
                col[s] = tensors[s] + keys[b * m + s];
                idx[s] = 0;
                if (last[s] < 0) pre *= col[s][0];   /* subcircuit with no cuts: plain factor */
            }
            out[b] = scale * rec(&c, 0, idx, pre);
        }
        free(idx);
        free((void *)col);
    }
    free(inc_sub); free(inc_str); free(fill); free(last); free(close_ofs); free(closes); free(pos);
    return used;
}
