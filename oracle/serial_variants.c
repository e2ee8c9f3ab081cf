/*
 * ORACLE-SIDE BASELINES -- TEST/BENCH INFRASTRUCTURE ONLY.  The paper's other serial Four-Russians variants
 * (section 3.2), single thread, column-wise fill as in Algorithm 1, timed on
 * the host beside the GPU for the speed-up table PAPER.md:313-323.  Each is pinned to eq. (1) like Algorithm 1
 * (tests/test_oracle_pins.py).  No code is shared with the CUDA path.
 *
 *   variant 1  partially memoised: "upon completion of elements of a group, if a new horizontal
 *              vector is seen, we pair it with all possible 2^q column vectors and the results are tabled".
 *   variant 2  completely memoised: "the result for a pair of vectors is computed the first time the
 *              pair is observed"; every lookup checks whether the pair has been processed.
 *   variant 3  Frid-Gusfield: after the q cells of a group in a row are computed, the black box
 *              is run for this fixed horizontal vector with all 2^q vertical vectors and D(i,p) is added; the table
 *              is indexed by row, group and (potential column) vector; the horizontal vectors are not stored.  To
 *              fill a cell the column vector of every group is looked up in that row's table and D(q,j) is added.
 *
 * The readings of Algorithm 1's loosely defined parts (g13-g16) and the vector encoding are those
 * of two_vector_serial.c.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

static int sv_code(uint8_t c)
{
    switch (c) {
    case 'A': case 'a': return 0;
    case 'C': case 'c': return 1;
    case 'G': case 'g': return 2;
    case 'U': case 'u': case 'T': case 't': return 3;
    default: return -1;
    }
}

/* the black box of PAPER.md:94-111: max over k of (prefix sum of v) + (prefix sum of vbar), from 0 */
static int sv_blackbox(int q, uint32_t v, uint32_t w)
{
    int maxval = 0, s1 = 0, s2 = 0;
    for (int k = 0; k < q; ++k) {
        s1 += (int)((v >> k) & 1u);
        s2 -= (int)((w >> k) & 1u);
        if (s1 + s2 > maxval) maxval = s1 + s2;
    }
    return maxval;
}

/*
 * Returns D(1,n) (-1 invalid base / bad arguments, -2 out of memory).  table_out (may be NULL): n x n row-major
 * int32, 0 below the diagonal.  stats (may be NULL): [0] table lookups in the group loop, [1] black-box
 * evaluations (preprocessing work), [2] bytes of the preprocessing table.
 */
int oracle_serial_variant(const uint8_t *seq, int n, int q, int variant, int32_t *table_out, int64_t *stats)
{
    if (n < 0 || q < 2 || q > 12 || variant < 1 || variant > 3) return -1;
    for (int t = 0; t < n; ++t) if (sv_code(seq[t]) < 0) return -1;
    if (stats) stats[0] = stats[1] = stats[2] = 0;
    if (n == 0) return 0;
    const size_t W = (size_t)n + 2;
    const size_t G = (size_t)n / q + 2;                  /* groups per row / column */
    const uint32_t N = 1u << q;
    int32_t *D = (int32_t *)calloc(W * W, sizeof(int32_t));
    uint16_t *hvec = (uint16_t *)calloc(W * G, sizeof(uint16_t));   /* [i][g] (not used by FG) */
    uint16_t *vvec = (uint16_t *)calloc(W * G, sizeof(uint16_t));   /* [j][g] */
    uint8_t *R = NULL;          /* variants 1, 2: R[v][w], 0xFF = not computed yet */
    uint8_t *rowdone = NULL;    /* variant 1: horizontal vector v has been paired with every w */
    int16_t *T = NULL;          /* variant 3: T[i][g][w] = D(i,gq) + max-val(v(i,g), w) */
    size_t tbytes = 0;
    if (variant == 3) { tbytes = W * G * N * sizeof(int16_t); T = (int16_t *)malloc(tbytes); }
    else { tbytes = (size_t)N * N; R = (uint8_t *)malloc(tbytes); rowdone = (uint8_t *)calloc(N, 1); }
    if (!D || !hvec || !vvec || (variant == 3 ? !T : (!R || !rowdone))) {
        free(D); free(hvec); free(vvec); free(R); free(rowdone); free(T);
        return -2;
    }
    if (R) memset(R, 0xFF, (size_t)N * N);
    int64_t lookups = 0, evals = 0;
#define DD(i, j) D[(size_t)(i) * W + (size_t)(j)]
    for (int j = 1; j <= n; ++j) {
        DD(j, j) = 0;
        for (int i = j - 1; i >= 1; --i) {
            int best = (sv_code(seq[i - 1]) + sv_code(seq[j - 1]) == 3) + DD(i + 1, j - 1);
            int gfirst = (i + q - 1) / q;
            int glast = j / q - 1;
            if (gfirst > glast) {
                for (int k = i + 1; k <= j; ++k) {
                    int c = DD(i, k - 1) + DD(k, j);
                    if (c > best) best = c;
                }
            } else {
                for (int k = i + 1; k <= gfirst * q; ++k) {
                    int c = DD(i, k - 1) + DD(k, j);
                    if (c > best) best = c;
                }
                for (int k = (glast + 1) * q + 1; k <= j; ++k) {
                    int c = DD(i, k - 1) + DD(k, j);
                    if (c > best) best = c;
                }
                for (int g = gfirst; g <= glast; ++g) {
                    const uint32_t w = vvec[(size_t)j * G + g];
                    int c;
                    if (variant == 3) {
                        /* the preprocessed value for this column vector in the row's block + D(q,j) */
                        c = T[((size_t)i * G + g) * N + w] + DD(g * q + 1, j);
                    } else {
                        const uint32_t v = hvec[(size_t)i * G + g];
                        uint8_t *e = &R[(size_t)v * N + w];
                        if (variant == 2 && *e == 0xFF) { *e = (uint8_t)sv_blackbox(q, v, w); ++evals; }
                        c = DD(i, g * q) + DD(g * q + 1, j) + *e;                                          /* eq. (3) */
                    }
                    if (c > best) best = c;
                }
                lookups += glast - gfirst + 1;
            }
            DD(i, j) = best;
            if (i % q == 1 % q) {                         /* vertical vector of row group (i-1)/q of column j */
                int g = (i - 1) / q;
                if (g * q + q <= j) {
                    uint32_t w = 0;
                    for (int p = 1; p < q; ++p)
                        w |= (uint32_t)(DD(g * q + p, j) - DD(g * q + 1 + p, j)) << p;
                    vvec[(size_t)j * G + g] = (uint16_t)w;
                }
            }
            if (j % q == q - 1) {                         /* the q cells of column group j/q of row i are complete */
                int g = j / q;
                if (g * q >= i) {
                    uint32_t v = 0;
                    for (int p = 1; p < q; ++p)
                        v |= (uint32_t)(DD(i, g * q + p) - DD(i, g * q + p - 1)) << p;
                    if (variant == 3) {                   /* all column vectors for this fixed v, + D(i,p) */
                        int16_t *row = &T[((size_t)i * G + g) * N];
                        const int anchor = DD(i, g * q);
                        for (uint32_t w = 0; w < N; ++w) row[w] = (int16_t)(anchor + sv_blackbox(q, v, w));
                        evals += N;
                    } else {
                        hvec[(size_t)i * G + g] = (uint16_t)v;
                        if (variant == 1 && !rowdone[v]) {    /* a new horizontal vector */
                            for (uint32_t w = 0; w < N; ++w) R[(size_t)v * N + w] = (uint8_t)sv_blackbox(q, v, w);
                            rowdone[v] = 1;
                            evals += N;
                        }
                    }
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
    if (stats) { stats[0] = lookups; stats[1] = evals; stats[2] = (int64_t)tbytes; }
    free(D); free(hvec); free(vvec); free(R); free(rowdone); free(T);
    return result;
}
