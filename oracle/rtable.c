/*
 * ORACLE -- TEST INFRASTRUCTURE ONLY.  The black-box evaluator of PAPER.md:91-111 (section 3.1)
 * and the table R built from it, written step by step in the paper's order.
 *
 *   Input: horizontal difference vector v (v_k in {0,1}) and vertical difference vector
 *          vbar (vbar_k in {0,-1}), both of length q.
 *   1: max-val <- 0 and max-index <- 0
 *   2: sum1 <- 0 and sum2 <- 0
 *   3: for k = 0 to q-1 do
 *   4:    sum1 <- sum1 + v_k          (the listing prints "v_i"; reading g11: the index is k)
 *   5:    sum2 <- sum2 + vbar_k
 *   6:    if sum1 + sum2 > max-val then
 *   7:       max-val <- sum1 + sum2
 *   8:       max-index <- k
 *   9:    end if
 *  10: end for
 *  11: return (max-val, max-index)
 *
 * Index convention (reading g12): a vector is the integer sum_k |v_k| 2^k, i.e. bit k
 * of the index is |v_k|.  R has 2^q x 2^q entries, "indexed by a pair of numbers in the range
 * [2^q]".  In the fill, v_0 = vbar_0 = 0 by definition, so only
 * even indices are reached; the loop is still well defined for every index and the whole table
 * is tabulated as the paper says ("all possible vector pairs of length q").
 */
#include <stdint.h>
#include <stddef.h>

int oracle_blackbox(int q, uint32_t v, uint32_t vbar, int *max_index_out)
{
    int max_val = 0, max_index = 0;
    int sum1 = 0, sum2 = 0;
    for (int k = 0; k <= q - 1; ++k) {
        sum1 = sum1 + (int)((v >> k) & 1u);          /* v_k in {0,1}      */
        sum2 = sum2 - (int)((vbar >> k) & 1u);       /* vbar_k in {0,-1}  */
        if (sum1 + sum2 > max_val) {
            max_val = sum1 + sum2;
            max_index = k;
        }
    }
    if (max_index_out) *max_index_out = max_index;
    return max_val;
}

/* R[v * 2^q + vbar] = max-val for every pair; q in 1..12 */
int oracle_rtable(int q, uint8_t *R)
{
    if (q < 1 || q > 12 || !R) return -1;
    uint32_t N = 1u << q;
    for (uint32_t v = 0; v < N; ++v)
        for (uint32_t w = 0; w < N; ++w)
            R[(size_t)v * N + w] = (uint8_t)oracle_blackbox(q, v, w, 0);
    return 0;
}
