/*
 * ORACLE -- TEST INFRASTRUCTURE ONLY.  Brute-force pins for the Nussinov oracle: two
 * enumerators that use NO dynamic programming and not the recurrence eq. (1).
 *
 * Definition enumerated: "Complimentary bases can be paired, i.e., A with U and
 * C with G.  A set of disjoint pairs is a matching.  The pairs in a matching must not cross,
 * i.e., if bases in positions i and j are paired and if bases k and l are paired, then either
 * they are nested, i.e., i < k < l < j or they are non-intersecting, i.e., i < j < k < l.  The
 * objective is to maximize the number of pairings under these constraints."
 */
#include <stdint.h>

static int bf_code(uint8_t c)
{
    switch (c) {
    case 'A': case 'a': return 0;
    case 'C': case 'c': return 1;
    case 'G': case 'g': return 2;
    case 'U': case 'u': case 'T': case 't': return 3;
    default: return -1;
    }
}
static int bf_comp(uint8_t x, uint8_t y) { int a = bf_code(x), b = bf_code(y); return a >= 0 && b >= 0 && a + b == 3; }

/* ---- enumerator 1: every matching of complementary bases, crossing test at the leaf ---- */
typedef struct { const uint8_t *s; int n; int partner[32]; int best; } bf_state;

static int bf_noncrossing(const bf_state *st)
{
    /* all pairs (i,j), (k,l) with i<k: nested i<k<l<j, or disjoint i<j<k<l; crossing is i<k<j<l */
    for (int i = 0; i < st->n; ++i) {
        int j = st->partner[i];
        if (j <= i) continue;
        for (int k = i + 1; k < st->n; ++k) {
            int l = st->partner[k];
            if (l <= k) continue;
            if (k < j && j < l) return 0;
        }
    }
    return 1;
}

static void bf_rec(bf_state *st, int p, int npairs)
{
    if (p == st->n) {
        if (npairs > st->best && bf_noncrossing(st)) st->best = npairs;
        return;
    }
    if (st->partner[p] != -1) { bf_rec(st, p + 1, npairs); return; }
    bf_rec(st, p + 1, npairs);                       /* p stays unpaired */
    for (int r = p + 1; r < st->n; ++r) {            /* p pairs with a later free base */
        if (st->partner[r] == -1 && bf_comp(st->s[p], st->s[r])) {
            st->partner[p] = r; st->partner[r] = p;
            bf_rec(st, p + 1, npairs + 1);
            st->partner[p] = -1; st->partner[r] = -1;
        }
    }
}

/* largest non-crossing complementary matching of seq[0..n), n <= 24 (practical: n <= 14) */
int oracle_brute_force_matchings(const uint8_t *seq, int n)
{
    if (n < 0 || n > 24) return -1;
    bf_state st; st.s = seq; st.n = n; st.best = 0;
    for (int t = 0; t < n; ++t) { if (bf_code(seq[t]) < 0) return -1; st.partner[t] = -1; }
    bf_rec(&st, 0, 0);
    return st.best;
}

/* ---- enumerator 2: structural recursion without memo: the first base of the interval is
 * unpaired, or pairs with position k and splits the rest into inside / outside (non-crossing
 * by construction).  A different decomposition from eq. (1) (which splits at an arbitrary k). */
static int bf_struct(const uint8_t *s, int lo, int hi)   /* interval [lo,hi] inclusive */
{
    if (lo >= hi) return 0;
    int best = bf_struct(s, lo + 1, hi);
    for (int k = lo + 1; k <= hi; ++k) {
        if (bf_comp(s[lo], s[k])) {
            int c = 1 + bf_struct(s, lo + 1, k - 1) + bf_struct(s, k + 1, hi);
            if (c > best) best = c;
        }
    }
    return best;
}

int oracle_brute_force_structural(const uint8_t *seq, int n)
{
    if (n < 0 || n > 20) return -1;
    for (int t = 0; t < n; ++t) if (bf_code(seq[t]) < 0) return -1;
    return bf_struct(seq, 0, n - 1);
}
