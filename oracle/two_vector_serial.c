/*
 * ORACLE-SIDE BASELINE -- TEST/BENCH INFRASTRUCTURE ONLY.  The paper's serial two-vector
 * Four-Russians method, Algorithm 1, single thread, column-wise fill.  It is
 * (a) the "serial two-vector CPU build" BASELINE.json asks to be timed on the host beside the
 * GPU, and (b) a pin that eq. (3) reproduces the plain table of eq. (1).
 * It is NOT the definitional oracle (that is nussinov.c) and shares no code with the CUDA path.
 *
 * Readings used: g13 column indices are grouped (0..q-1),(q..2q-1),... and row
 * indices (1..q),(q+1..2q),...; g14 full groups of cell (i,j) are
 * g = ceil(i/q) .. floor(j/q)-1, head residual k = i+1 .. ceil(i/q)*q, tail residual
 * k = floor(j/q)*q+1 .. j, plain loop if there is no full group; g15 "D(i,p)+D(q,j)" is the row
 * anchor D(i,gq) plus the column anchor D(gq+1,j) of the same group; g16 the vertical vector of
 * group g in column j is stored when cell (gq+1,j) is done and the horizontal vector of group g
 * in row i when cell (i,gq+q-1) is done.
 *
 * Vector encoding: v_0 = 0, v_p = D(i,l+p) - D(i,l+p-1) in {0,1};
 * vbar_0 = 0, vbar_p = D(l+1+p,j) - D(l+p,j) in {0,-1}; index = sum_p |v_p| 2^p.
 */
#include <stdint.h>
#include <stdlib.h>

static int tv_code(uint8_t c)
{
    switch (c) {
    case 'A': case 'a': return 0;
    case 'C': case 'c': return 1;
    case 'G': case 'g': return 2;
    case 'U': case 'u': case 'T': case 't': return 3;
    default: return -1;
    }
}

/* line 1 of Algorithm 1: R <- preprocess all pairs of vectors of length q */
static void tv_preprocess(int q, uint8_t *R)
{
    uint32_t N = 1u << q;
    for (uint32_t v = 0; v < N; ++v)
        for (uint32_t w = 0; w < N; ++w) {
            int maxval = 0, s1 = 0, s2 = 0;
            for (int k = 0; k < q; ++k) {
                s1 += (int)((v >> k) & 1u);
                s2 -= (int)((w >> k) & 1u);
                if (s1 + s2 > maxval) maxval = s1 + s2;
            }
            R[(size_t)v * N + w] = (uint8_t)maxval;
        }
}

/*
 * Returns D(1,n) (or -1 invalid base / bad q, -2 out of memory).  table_out (may be NULL):
 * n x n row-major int32, 0 below the diagonal.  lookups_out (may be NULL): number of R lookups.
 */
int oracle_two_vector_serial(const uint8_t *seq, int n, int q, int32_t *table_out, int64_t *lookups_out)
{
    if (n < 0 || q < 2 || q > 12) return -1;
    for (int t = 0; t < n; ++t) if (tv_code(seq[t]) < 0) return -1;
    if (n == 0) { if (lookups_out) *lookups_out = 0; return 0; }
    size_t W = (size_t)n + 2;
    size_t G = (size_t)n / q + 2;                    /* groups per row / column */
    uint32_t N = 1u << q;
    int32_t *D = (int32_t *)calloc(W * W, sizeof(int32_t));
    uint16_t *hvec = (uint16_t *)calloc(W * G, sizeof(uint16_t));   /* [i][g] */
    uint16_t *vvec = (uint16_t *)calloc(W * G, sizeof(uint16_t));   /* [j][g] */
    uint8_t *R = (uint8_t *)malloc((size_t)N * N);
    if (!D || !hvec || !vvec || !R) { free(D); free(hvec); free(vvec); free(R); return -2; }
    tv_preprocess(q, R);                                            /* line 1 */
    int64_t lookups = 0;
#define DD(i, j) D[(size_t)(i) * W + (size_t)(j)]
    for (int j = 1; j <= n; ++j) {                                  /* line 2 */
        DD(j, j) = 0;                                               /* line 3 */
        for (int i = j - 1; i >= 1; --i) {                          /* line 4 */
            int best = (tv_code(seq[i - 1]) + tv_code(seq[j - 1]) == 3) + DD(i + 1, j - 1);  /* line 5 */
            int gfirst = (i + q - 1) / q;                           /* lines 6-8, reading g14 */
            int glast = j / q - 1;
            if (gfirst > glast) {
                for (int k = i + 1; k <= j; ++k) {                  /* no full group: plain */
                    int c = DD(i, k - 1) + DD(k, j);
                    if (c > best) best = c;
                }
            } else {
                for (int k = i + 1; k <= gfirst * q; ++k) {         /* lines 9-11: first group */
                    int c = DD(i, k - 1) + DD(k, j);
                    if (c > best) best = c;
                }
                for (int k = (glast + 1) * q + 1; k <= j; ++k) {    /* lines 12-14: last group */
                    int c = DD(i, k - 1) + DD(k, j);
                    if (c > best) best = c;
                }
                for (int g = gfirst; g <= glast; ++g) {             /* lines 15-19: groups in between */
                    int c = DD(i, g * q) + DD(g * q + 1, j)
                          + R[(size_t)hvec[(size_t)i * G + g] * N + vvec[(size_t)j * G + g]];   /* eq. (3) */
                    if (c > best) best = c;
                }
                lookups += glast - gfirst + 1;
            }
            DD(i, j) = best;
            /* lines 20-22: vertical vector of row group g = (i-1)/q (rows gq+1..gq+q) of column j */
            if (i % q == 1 % q) {
                int g = (i - 1) / q;
                if (g * q + q <= j) {
                    uint32_t w = 0;
                    for (int p = 1; p < q; ++p)
                        w |= (uint32_t)(DD(g * q + p, j) - DD(g * q + 1 + p, j)) << p;   /* |vbar_p| */
                    vvec[(size_t)j * G + g] = (uint16_t)w;
                }
            }
            /* lines 23-25: horizontal vector of column group g = j/q (columns gq..gq+q-1) of row i */
            if (j % q == q - 1) {
                int g = j / q;
                if (g * q >= i) {
                    uint32_t v = 0;
                    for (int p = 1; p < q; ++p)
                        v |= (uint32_t)(DD(i, g * q + p) - DD(i, g * q + p - 1)) << p;   /* v_p */
                    hvec[(size_t)i * G + g] = (uint16_t)v;
                }
            }
        }
    }
    int result = DD(1, n);
    if (table_out)
        for (int i = 1; i <= n; ++i)
            for (int j = 1; j <= n; ++j)
                table_out[(size_t)(i - 1) * n + (j - 1)] = (j >= i) ? DD(i, j) : 0;
#undef DD
    if (lookups_out) *lookups_out = lookups;
    free(D); free(hvec); free(vvec); free(R);
    return result;
}
