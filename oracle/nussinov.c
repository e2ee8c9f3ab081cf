/*
 * ORACLE -- TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct CPU implementation of
 * what the hot path computes.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call this.  It shares no code with the CUDA path.
 *
 * What it computes (section 2, eq. (1)):
 *   S[1..n] over {A,C,G,U};  D(i,i-1) = D(i,i) = 0 for all i;  for i < j
 *     D(i,j) = max{ b(S_i,S_j) + D(i+1,j-1),  max_{i+1<=k<=j} D(i,k-1) + D(k,j) }
 *   b = 1 for complementary bases (A-U, C-G), else 0.  Result D(1,n).
 * Readings: g1 Watson-Crick pairs only (no G-U wobble,
 * PAPER.md:45 "A with U and C with G"); g2 no minimum hairpin loop (eq. (1) lets adjacent
 * bases pair); g3 D(i,i-1)=0 exists for i=1..n+1; g4 upper/lower case accepted, T==U, any
 * other byte is an error (-1).
 *
 * The method under test (two-vector Four-Russians) reaches EXACTLY this table (eq. (3) is an
 * identity), so the oracle is the plain definition: triple loop, int32, no
 * grouping, no lookup.  Parity: pinned (tests/test_oracle_pins.py: brute-force enumeration,
 * hand-worked values, closed forms, invariants, symmetries).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* base byte -> code 0..3 (A,C,G,U), -1 otherwise (reading g4) */
static int base_code(uint8_t c)
{
    switch (c) {
    case 'A': case 'a': return 0;
    case 'C': case 'c': return 1;
    case 'G': case 'g': return 2;
    case 'U': case 'u': case 'T': case 't': return 3;
    default: return -1;
    }
}

/* b(x,y) of eq. (1): 1 iff {x,y} = {A,U} or {C,G} */
static int pair_score(int x, int y)
{
    return (x + y == 3) ? 1 : 0;   /* A=0,U=3 ; C=1,G=2 */
}

int oracle_validate(const uint8_t *seq, int n)
{
    for (int t = 0; t < n; ++t)
        if (base_code(seq[t]) < 0) return -1;
    return 0;
}

/*
 * Plain Nussinov, eq. (1), filled by diagonals ("(i,i)-diagonal first,
 * (i,i+1)-diagonal next and so on").  table_out (may be NULL) receives the n x n row-major
 * table: entry [i-1][j-1] = D(i,j) for i<=j, 0 below the diagonal.  Returns D(1,n), or -1
 * for an invalid base.  n = 0 and n = 1 give 0.
 */
int oracle_nussinov(const uint8_t *seq, int n, int32_t *table_out)
{
    if (n < 0 || oracle_validate(seq, n) != 0) return -1;
    if (n == 0) return 0;
    /* D indexed [i][j], i in 1..n+1, j in 0..n; calloc gives D(i,i-1) = D(i,i) = 0 */
    size_t W = (size_t)n + 2;
    int32_t *D = (int32_t *)calloc(W * W, sizeof(int32_t));
    if (!D) return -2;
#define DD(i, j) D[(size_t)(i) * W + (size_t)(j)]
    for (int d = 1; d <= n - 1; ++d) {             /* d = j - i */
        for (int i = 1; i + d <= n; ++i) {
            int j = i + d;
            int best = pair_score(base_code(seq[i - 1]), base_code(seq[j - 1])) + DD(i + 1, j - 1);
            for (int k = i + 1; k <= j; ++k) {
                int c = DD(i, k - 1) + DD(k, j);
                if (c > best) best = c;
            }
            DD(i, j) = best;
        }
    }
    int result = DD(1, n);
    if (table_out) {
        for (int i = 1; i <= n; ++i)
            for (int j = 1; j <= n; ++j)
                table_out[(size_t)(i - 1) * n + (j - 1)] = (j >= i) ? DD(i, j) : 0;
    }
#undef DD
    free(D);
    return result;
}

/*
 * The same table by the four-term form BASELINE.json's north_star writes:
 *   S(i,j) = max{ S(i+1,j), S(i,j-1), S(i+1,j-1)+b(i,j), max_{i<=k<j} S(i,k)+S(k+1,j) }.
 * Equal to eq. (1) (substitute k' = k-1; the end terms are D(i+1,j) and D(i,j-1)); kept so a
 * test can assert the equality instead of trusting the algebra.
 */
int oracle_nussinov_fourterm(const uint8_t *seq, int n, int32_t *table_out)
{
    if (n < 0 || oracle_validate(seq, n) != 0) return -1;
    if (n == 0) return 0;
    size_t W = (size_t)n + 2;
    int32_t *D = (int32_t *)calloc(W * W, sizeof(int32_t));
    if (!D) return -2;
#define DD(i, j) D[(size_t)(i) * W + (size_t)(j)]
    for (int d = 1; d <= n - 1; ++d) {
        for (int i = 1; i + d <= n; ++i) {
            int j = i + d;
            int best = DD(i + 1, j);
            if (DD(i, j - 1) > best) best = DD(i, j - 1);
            int p = DD(i + 1, j - 1) + pair_score(base_code(seq[i - 1]), base_code(seq[j - 1]));
            if (p > best) best = p;
            for (int k = i; k < j; ++k) {
                int c = DD(i, k) + DD(k + 1, j);
                if (c > best) best = c;
            }
            DD(i, j) = best;
        }
    }
    int result = DD(1, n);
    if (table_out) {
        for (int i = 1; i <= n; ++i)
            for (int j = 1; j <= n; ++j)
                table_out[(size_t)(i - 1) * n + (j - 1)] = (j >= i) ? DD(i, j) : 0;
    }
#undef DD
    free(D);
    return result;
}

/*
 * "fast-plain" mode: the SAME recurrence eq. (1), same diagonal order, same k range; the only
 * change is storage: besides the row-major table Rw[i][c] = D(i,c) a transposed mirror
 * Mr[j][k] = D(k,j) is kept (the public idea PAPER.md:285 attributes to Chang et al. [6]), so
 * the k loop reads two contiguous int16 arrays and the compiler can vectorise it.  The cells of
 * one diagonal are independent, so they may be split over `threads` OpenMP
 * threads.  Validated cell by cell against oracle_nussinov (tests/test_oracle_pins.py); used
 * for the n = 6000 and n = 16384 expected values.  int16 is exact for n <= 65534.
 *
 * cells: `ncells` pairs (i,j), 1-based, i<=j -> cell_values[t] = D(i,j).
 * table_out16 (may be NULL): n x n row-major int16, 0 below the diagonal.
 * table_sum (may be NULL): sum over i<=j of D(i,j).
 */
int oracle_nussinov_fast(const uint8_t *seq, int n, int threads,
                         const int32_t *cells, int ncells, int32_t *cell_values,
                         int16_t *table_out16, int64_t *table_sum)
{
    if (n < 0 || n > 65534 || oracle_validate(seq, n) != 0) return -1;
    if (n == 0) { if (table_sum) *table_sum = 0; return 0; }
    size_t W = (size_t)n + 2;
    int16_t *Rw = (int16_t *)calloc(W * W, sizeof(int16_t));
    int16_t *Mr = (int16_t *)calloc(W * W, sizeof(int16_t));
    int8_t *code = (int8_t *)malloc((size_t)n + 2);
    if (!Rw || !Mr || !code) { free(Rw); free(Mr); free(code); return -2; }
    for (int t = 1; t <= n; ++t) code[t] = (int8_t)base_code(seq[t - 1]);
    if (threads < 1) threads = 1;
    for (int d = 1; d <= n - 1; ++d) {
#pragma omp parallel for num_threads(threads) schedule(static)
        for (int i = 1; i <= n - d; ++i) {
            int j = i + d;
            const int16_t *row = Rw + (size_t)i * W;     /* row[c] = D(i,c)  */
            const int16_t *col = Mr + (size_t)j * W;     /* col[k] = D(k,j)  */
            int16_t best = (int16_t)(pair_score(code[i], code[j]) + Rw[(size_t)(i + 1) * W + (j - 1)]);
            for (int k = i + 1; k <= j; ++k) {
                int16_t c = (int16_t)(row[k - 1] + col[k]);
                best = c > best ? c : best;
            }
            Rw[(size_t)i * W + j] = best;
            Mr[(size_t)j * W + i] = best;
        }
    }
    int result = Rw[(size_t)1 * W + n];
    for (int t = 0; t < ncells; ++t) {
        int i = cells[2 * t], j = cells[2 * t + 1];
        cell_values[t] = (i >= 1 && j <= n && i <= j) ? Rw[(size_t)i * W + j] : -1;
    }
    if (table_sum) {
        int64_t s = 0;
        for (int i = 1; i <= n; ++i)
            for (int j = i; j <= n; ++j) s += Rw[(size_t)i * W + j];
        *table_sum = s;
    }
    if (table_out16) {
        for (int i = 1; i <= n; ++i)
            for (int j = 1; j <= n; ++j)
                table_out16[(size_t)(i - 1) * n + (j - 1)] = (j >= i) ? Rw[(size_t)i * W + j] : 0;
    }
    free(Rw); free(Mr); free(code);
    return result;
}
