// smem_engine.cuh -- RNA4R_ENGINE_SMEM: one CTA per sequence, the whole fold resident in shared memory.
//
// The engine for batches of short sequences (BASELINE.json configs[3]; north_star "batch many sequences to fill the
// machine on short diagonals").  Same coordinates and the same two-vector step as
// tiled_engine.cuh: M(r,c) = D(r+1,c), group g = split indices t in [gq, gq+q), and for row r, column c
//     max_{t in g} M(r,t) + M(t,c) = M(r,gq) + M(gq,c) + Rc[h][v]                     (eq. (3))
// with h / v the q-1 informative difference bits of the row run / the column run (v_0 = 0).
//
// What is stored ("only the horizontal and vertical differences are stored", plus anchors, reading g21):
//   W[A][j][a]   row word of row Aq+a over group g = A+1+j, 32 bit:  h << 24 | M(r,gq)      (tile-row major)
//   X[B][g][y]   column word of column Bq+y over group g <= B, 16 bit:  v << (16-HB) | M(gq,c); expanded on load to
//                v << (24-HB) | M(gq,c), so that S = W + X has the table index h*2^HB + v at bit 24-HB and the
//                anchor sum in the low halfword: one lookup = add, LEA.HI, LDS.U8, VIADDMNMX.U16x2.
// Nothing else of the table is kept: n^2/(2q) words of each kind (n = 700, q = 8: 122 KB + 61 KB).  Both arrays are
// laid out so that the groups a row block / a column meets one after another are a constant stride apart.
//
// Schedule.  q x q tiles (A,B); the tiles of one tile-diagonal D = B - A are independent.  For a tile
// the groups strictly between A and B are complete for all its q^2 cells (Alg. 1 lines 15-19);
// groups A and B are the paper's residual loops.  One CTA barrier per tile-diagonal step D; the
// warps share, dealt round-robin,
//   (i)  the waves: the closure of every tile of diagonal D, 4 tiles per warp (Q lanes each), and
//   (ii) the bulk of diagonal D+1 and later: for every strip-tile (tile-row A x 4 tile-columns = 32 columns) whose
//        first tile lies on diagonal D0 = D+1, the complete groups j = g-A-1 in [1, D0-3] that no tile of diagonal D
//        feeds -- lanes <-> 32 columns of ONE row, so the row word is warp-uniform and the table gather is conflict-
//        free.  The maxima are packed into one word per column (value of the bottom row + 3-bit offsets of the rows
//        above: Lemma 1 bounds them by q-1) in a 5-slot ring per tile-row.
// The groups a strip-tile cannot take yet ("fresh": j in [0,k] and [D0-2, D-2] for its k-th tile column, at most
// 4 per side) are looked up inside the wave.
//
// Wave of tile (A,B), row-parallel: rows from the bottom up, the Q cells of a row at once.  With
//   C'(a,y) = max{ bulk, fresh, b + M(r+1,c-1), head: max_{t in group A, t>r} M(r,t)+M(t,c) }   -- rows below only
// the row is  V(a,y) = max_{y' <= y} C'(a,y') + Qd(y',y),  Qd = the diagonal tile (B,B): the in-row dependency
// V(a,y) >= V(a,y') + Qd(y',y) collapses because Qd is superadditive (M(i,k) >= M(i,j) + M(j,k)).  The head is one
// masked lookup with the running column word; the tail is a max-plus over the row's packed C' values
// (4 DPX VIADDMNMX.S16x2).  No skewed wavefront: 8 dependent steps per tile, every lane busy in every step.
#pragma once
#include <new>
#include <type_traits>
#include "common.cuh"

namespace smemseq {

template <int Q>
struct Cfg {
    static_assert(Q >= 4 && Q <= 8, "the shared-memory engine is built for q = 4..8");
    static constexpr int HB = Q - 1;                 // informative bits per vector
    static constexpr int G = 4;                      // q-tiles per warp and per column strip
    static constexpr int SW = G * Q;                 // strip width in columns (<= 32)
    static constexpr int ISH = 24 - HB;              // position of the table index in a word sum
    static constexpr int XAB = 16 - HB;              // anchor bits of a stored column word
    static constexpr uint32_t XAMASK = (1u << XAB) - 1u;
    static constexpr uint32_t XMUL = (1u << ISH) - (1u << XAB);
    static constexpr uint32_t HMASK = (1u << HB) - 1u;
    static constexpr int TBL_BYTES = 1 << (2 * HB);
    static constexpr int TBL_AREA = TBL_BYTES < 256 ? 256 : TBL_BYTES;
#ifndef RNA4R_SMEM_NWARP
#define RNA4R_SMEM_NWARP 24
#endif
    static constexpr int NWARP = RNA4R_SMEM_NWARP;   // 80 registers per thread x 768 threads: the register file of one SM
    static constexpr int NTHR = NWARP * 32;
    static constexpr int NP = (Q + 1) / 2;           // packed value pairs of a tile row
    static constexpr int VBITS = 11;                 // value bits of a packed bulk word (D <= 2047)
    static constexpr int VPITCH = 40;                // words per tile-row of the bulk ring: 5 tile-column slots x 8
    static constexpr int SCR_WARP_HW = 2 * G * 8 + 8 * 2 + 8;    // per-warp scratch in halfwords: row buffers [2][G][8], two dummy store targets
    static constexpr int SCR_BYTES = NWARP * SCR_WARP_HW * 2;
    static constexpr int FIXED_BYTES = TBL_AREA + SCR_BYTES + 64;
#ifndef RNA4R_SMEM_DATAFLOW
#define RNA4R_SMEM_DATAFLOW 0
#endif
    // Build knob: progress words per tile-row (waves wait for their two neighbours, bulk tasks for a complete diagonal)
    // instead of the CTA barrier per tile-diagonal.  Measured equal (cfg4 1.60 vs 1.59 ms): the barrier is not what a
    // sequence waits for, the chain of waves through its neighbours is.
    static constexpr bool DATAFLOW = RNA4R_SMEM_DATAFLOW != 0;
#ifndef RNA4R_SMEM_TOPUP
#define RNA4R_SMEM_TOPUP 1
#endif
    // top-up tasks: the groups a strip-tile's bulk pass had to leave out for its later tile columns (they were not
    // finished yet) are looked up one step before the tile closes, off the wave's path; the wave keeps two fresh groups
    static constexpr bool TOPUP = !DATAFLOW && RNA4R_SMEM_TOPUP != 0;
    static constexpr int MAX_SMEM = 232448;          // 227 KB
};

// byte offsets of one sequence's state, relative to the start of the pool
struct Layout {
    int NB;
    uint32_t W, X, val, wdh, dq, pm, rl, code, plan, flags, total;
};

template <int Q>
__host__ __device__ inline Layout make_layout(int n)
{
    Layout L;
    const uint32_t NB = (uint32_t)(n / Q + 1);
    L.NB = (int)NB;
    uint32_t off = 0;
    auto take = [&](uint32_t bytes) { const uint32_t o = off; off += (bytes + 15u) & ~15u; return o; };
    L.W = take(4u * Q * NB * (NB - 1) / 2);
    L.X = take(2u * Q * NB * (NB + 1) / 2);
    L.val = take(4u * Cfg<Q>::VPITCH * (NB + 1));
    L.wdh = take(4u * Q * NB);
    L.dq = take(8u * Q * NB);
    L.pm = take(4u * NB);
    L.rl = take(2u * Q * NB);
    L.code = take(Q * NB + 16u);
    L.plan = take(4u * NB);
    L.flags = take(4u * (3u * NB + 8u));
    L.total = off;
    return L;
}

// largest n this engine folds: the state has to fit the pool, the anchors their fields
template <int Q>
inline int max_n()
{
    const uint32_t pool = (uint32_t)(Cfg<Q>::MAX_SMEM - Cfg<Q>::FIXED_BYTES);
    int lim = 2 * ((1 << Cfg<Q>::XAB) - 1);                         // D <= n/2 < 2^XAB
    if (lim > 2 * ((1 << Cfg<Q>::VBITS) - 1)) lim = 2 * ((1 << Cfg<Q>::VBITS) - 1);
    int lo = 0, hi = lim;
    while (lo < hi) {
        const int mid = (lo + hi + 1) / 2;
        if (make_layout<Q>(mid).total <= pool) lo = mid; else hi = mid - 1;
    }
    return lo;
}

struct Params {
    const uint8_t *seqs;
    const int64_t *offsets;   // device [count+1], or NULL for a single sequence of length n_single
    const int32_t *lens;      // device [count] (batch only)
    const int32_t *order;     // device [grid]: sequence folded by CTA b (longest first), or NULL: CTA b folds b
    int n_single;
    const uint8_t *tbl;       // compact table Rc, bytes, natural pitch
    int32_t *scores;
    int32_t *status;          // NULL or [count]
    void *table_out;          // NULL, or n*n elements (single sequence only)
    int table_dtype;
    unsigned long long *trace;   // NULL, or [trace_seqs][8] clock64 sums of warp 0 (rna4r_set_trace): total, setup + diagonal
    int trace_seqs;              // tiles, waves + bulk, merge phases, wave tasks, #wave tasks, bulk tasks, n
};

template <int Q>
struct Sm {
    uint32_t tbl_sa;          // shared-space address of the table
    uint16_t *scr;            // per-warp row scratch
    int *misc;                // [1] invalid flag
    uint32_t *W;
    uint16_t *X;
    uint32_t *val;
    uint32_t *wdh;
    uint8_t *dq;
    uint8_t *pm;
    int16_t *rl;
    int8_t *code;
    uint32_t *plan;           // [NB] step_plan of every tile-diagonal
    int *prog;                // [NB+1] last tile-diagonal tile-row A has finished          (dataflow schedule)
    int *bulkd;               // [NB+1] first diagonal D0 of the last strip-tile whose bulk word is in the ring
    int *cntd;                // [NB+1] finished tiles per tile-diagonal; cntd[NB+1] = last tile-diagonal that is complete
    int n, NB;
};

__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// acc = max(acc, candidate of the word sum S): eq. (3).  No mask on the index: a don't-care S of an
// idle lane indexes at most 2^(8+HB) bytes past the table, inside the CTA's window (the pool follows the table).
template <int Q>
__device__ __forceinline__ uint32_t lookup_max(uint32_t tbl_sa, uint32_t S, uint32_t acc)
{
    uint32_t rv;
    asm("ld.shared.u8 %0, [%1];" : "=r"(rv) : "r"((S >> Cfg<Q>::ISH) + tbl_sa));
    RNA4R_CHECK((S >> Cfg<Q>::ISH) < (uint32_t)Cfg<Q>::TBL_BYTES && (S & 0xffffu) + rv < (1u << Cfg<Q>::VBITS));
    return __viaddmax_u16x2(S, rv, acc);
}

template <int Q>
__device__ __forceinline__ uint32_t expand_x(uint32_t x16) { return x16 + (x16 >> Cfg<Q>::XAB) * Cfg<Q>::XMUL; }

template <int Q> __device__ __forceinline__ int off_w(int NB, int A) { return Q * (A * (NB - 1) - A * (A - 1) / 2); }   // words
template <int Q> __device__ __forceinline__ int off_x(int B) { return Q * (B * (B + 1) / 2); }                          // halfwords

// the Q row words of tile-row A over one group (warp- or tile-uniform address: broadcast loads)
template <int Q>
__device__ __forceinline__ void load_rows(const uint32_t *w, uint32_t (&wr)[Q])
{
    if constexpr (Q % 4 == 0) {
#pragma unroll
        for (int i = 0; i < Q / 4; ++i) {
            const uint4 t = reinterpret_cast<const uint4 *>(w)[i];
            wr[4 * i] = t.x; wr[4 * i + 1] = t.y; wr[4 * i + 2] = t.z; wr[4 * i + 3] = t.w;
        }
    } else {
#pragma unroll
        for (int a = 0; a < Q; ++a) wr[a] = w[a];
    }
}

// step a8 for the test / inspection path: out[(i-1)*n + (j-1)] = D(i,j) = M(i-1, j)
template <bool TABLE>
__device__ __forceinline__ void store_cell(const Params &p, int n, int r, int c, int v)
{
    if constexpr (TABLE) {
        if (r < n && c >= r + 1 && c <= n) {
            if (p.table_dtype == RNA4R_TABLE_INT16) reinterpret_cast<int16_t *>(p.table_out)[(size_t)r * n + c - 1] = (int16_t)v;
            else reinterpret_cast<int32_t *>(p.table_out)[(size_t)r * n + c - 1] = v;
        }
    }
}

// Bulk maxima of one column, packed: value of the bottom row | 3-bit offsets of the rows above.  All candidates of a
// strip-tile range over the same splits t, and M(r,t) - M(r_bottom,t) lies in [0, Q-1] (Lemma 1), so
// the maxima of the rows differ from the bottom row's by 0..Q-1.
template <int Q>
__device__ __forceinline__ uint32_t pack_rows(const uint32_t (&acc)[Q])
{
    const uint32_t base = acc[Q - 1] & 0xffffu;
    uint32_t w = base;
#pragma unroll
    for (int a = 0; a < Q - 1; ++a) {
        RNA4R_CHECK((acc[a] & 0xffffu) - base <= 7u && base < (1u << Cfg<Q>::VBITS));
        w |= (((acc[a] & 0xffffu) - base) & 7u) << (Cfg<Q>::VBITS + 3 * a);
    }
    return w;
}
template <int Q>
__device__ __forceinline__ int unpack_row(uint32_t w, int a)
{
    const int base = (int)(w & ((1u << Cfg<Q>::VBITS) - 1u));
    return a == Q - 1 ? base : base + (int)((w >> (Cfg<Q>::VBITS + 3 * a)) & 7u);
}

// ---- bulk (step a4): rows of tile-row A x the 32 columns of the strip that starts at tile column GC -----------------
// Groups j = g-A-1 in [jlo, jhi] (1 <= jlo).  lane <-> column, a thread owns the Q rows; the row words are warp-uniform
// (broadcast loads), so all 32 gathers of a lookup fall in one table row: conflict-free.  Group j of the strip's k-th
// tile column comes from tile (A+1+j, GC+k), which is finished only if j > k: the lanes of later tile columns sit
// out j = 1..3 (their share is looked up in the wave).
template <int Q>
__device__ __forceinline__ void strip_bulk(const Sm<Q> &s, int A, int GC, int jlo, int jhi, int lane, uint32_t (&acc)[Q])
{
    using C = Cfg<Q>;
    const int l2 = lane < C::SW ? lane : C::SW - 1;
    const int kq = l2 / Q, y = l2 - kq * Q;
    const int Bc = min(GC + kq, s.NB - 1);
    const uint32_t *w = s.W + off_w<Q>(s.NB, A) + jlo * Q;
    const uint16_t *x = s.X + off_x<Q>(Bc) + (A + 1 + jlo) * Q + y;
    int j = jlo;
    for (; j <= jhi && j <= C::G - 1; ++j) {
        const uint32_t X32 = (kq < j) ? expand_x<Q>(*x) : 0u;             // X = 0: a valid lower bound, nothing read
        uint32_t wr[Q];
        load_rows<Q>(w, wr);
#pragma unroll
        for (int a = 0; a < Q; ++a) acc[a] = lookup_max<Q>(s.tbl_sa, wr[a] + X32, acc[a]);
        w += Q; x += Q;
    }
#pragma unroll 4
    for (; j <= jhi; ++j) {
        const uint32_t X32 = expand_x<Q>(*x);
        uint32_t wr[Q];
        load_rows<Q>(w, wr);
#pragma unroll
        for (int a = 0; a < Q; ++a) acc[a] = lookup_max<Q>(s.tbl_sa, wr[a] + X32, acc[a]);
        w += Q; x += Q;
    }
}

// ring slot of (tile-row A, tile column Bc, column y) in the packed bulk maxima
template <int Q>
__device__ __forceinline__ int val_index(int A, int Bc, int y) { return A * Cfg<Q>::VPITCH + (Bc % 5) * 8 + y; }

// ---- diagonal tile (A,A): plain eq. (1) on Q x Q cells, one thread --------------------------------------------------
template <int Q, bool TABLE>
__device__ void diag_tile(const Params &p, const Sm<Q> &s, int seq, int A)
{
    using C = Cfg<Q>;
    const int r0 = A * Q;
    int m[Q][Q];
    int cd[Q];
#pragma unroll
    for (int a = 0; a < Q; ++a) {
        cd[a] = s.code[r0 + a];
#pragma unroll
        for (int y = 0; y < Q; ++y) m[a][y] = 0;
    }
#pragma unroll
    for (int d = 2; d < Q; ++d) {
#pragma unroll
        for (int a = 0; a + d < Q; ++a) {
            const int y = a + d;
            int best = m[a + 1][y - 1] + rna4r_pair(cd[a], cd[y - 1]);      // b(S_i,S_j) + D(i+1,j-1)
#pragma unroll
            for (int t = a + 1; t < y; ++t) best = max(best, m[a][t] + m[t][y]);
            m[a][y] = best;
        }
    }
    uint16_t *xo = s.X + off_x<Q>(A) + A * Q;
#pragma unroll
    for (int y = 0; y < Q; ++y) {
        uint32_t vb = 0;
#pragma unroll
        for (int j = 1; j < Q; ++j) vb |= (uint32_t)(m[j - 1][y] - m[j][y]) << (j - 1);
        xo[y] = (uint16_t)((vb << C::XAB) | (uint32_t)m[0][y]);
        uint8_t *dq = s.dq + (size_t)(r0 + y) * 8;
#pragma unroll
        for (int t = 0; t < 8; ++t) dq[t] = (t < Q && t < y) ? (uint8_t)m[t][y] : (uint8_t)0;
    }
#pragma unroll
    for (int a = 0; a < Q; ++a) {
        uint32_t hb = 0;
#pragma unroll
        for (int j = 1; j < Q; ++j) hb |= (uint32_t)(m[a][j] - m[a][j - 1]) << (j - 1);
        s.wdh[r0 + a] = hb << 24;
        s.rl[r0 + a] = (int16_t)m[a][Q - 1];
        if constexpr (TABLE) {
#pragma unroll
            for (int y = 0; y < Q; ++y) store_cell<TABLE>(p, s.n, r0 + a, r0 + y, m[a][y]);
        }
    }
    if (A == 0 && s.n < Q) {
        int v = 0;
#pragma unroll
        for (int y = 0; y < Q; ++y) if (y == s.n) v = m[0][y];
        p.scores[seq] = v;                                                   // M(0,n) = D(1,n)
    }
}

// ---- wave: closure of up to G tiles of tile-diagonal D --------------------------------------------------------------
// Task t = 4*jt + rho takes the tiles A = rho + 16*jt + 4*i, i = 0..3 (lane group i): they share k = (A + D) mod 4
// and D0 = D - k (the diagonal their strip-tile starts on), so every loop bound below is warp-uniform.
template <int Q, bool TABLE>
__device__ __forceinline__ void wave_task(const Params &p, const Sm<Q> &s, int seq, int D, int t, int warp, int lane)
{
    using C = Cfg<Q>;
    constexpr uint32_t FULL = 0xffffffffu;
    const int NB = s.NB, NT = NB - D;
    const int A0 = (t & 3) + 16 * (t >> 2);
    if (A0 >= NT) return;
    const bool lane_ok = lane < C::SW;
    const int i = lane_ok ? lane / Q : C::G - 1;
    const int y = lane_ok ? lane - i * Q : Q - 1;
    int A = A0 + C::G * i;
    const bool own = lane_ok && A < NT;
    if (A >= NT) A = A0;                                       // shadow of the first tile: computes, stores nothing
    const int B = A + D;
    const int k = B & (C::G - 1), D0 = D - k;
    const int r0 = A * Q, c = B * Q + y;
    const uint16_t *xcol = s.X + off_x<Q>(B) + y;              // xcol[g*Q] = column word of (group g, my column)
    const uint32_t *wrow = s.W + off_w<Q>(NB, A);              // wrow[j*Q + a] = row word of (row r0+a, group A+1+j)

    if constexpr (C::DATAFLOW) {
        // wait until my tile-row and the one below have finished tile-diagonal D-1 (every other operand of the tile is
        // older: each tile waited for the tile below it) and the strip-tile's bulk word has been written
        volatile int *pg = s.prog, *bd = s.bulkd;
        while (!__all_sync(FULL, pg[A] >= D - 1 && pg[A + 1] >= D - 1 && (D0 < 4 || bd[A] >= D0))) __nanosleep(32);
        __threadfence_block();
    }
    // Operands that do not depend on the fresh lookups are requested first: their shared-memory latency passes while
    // the fresh loop runs (a single warp issues in order).  Bulk maxima of the strip-tile (written during step D0 - 1;
    // none if the strip-tile starts before diagonal 4), the diagonal tile (B,B), the code of my column, the bottom edge
    // M((A+1)q, c) = anchor of the column word of group A+1, and the left column M(r0+1+y, Bq-1) for lane 0's pair term:
    // the last value tile (A,B-1) left in its rows, and for the row below the tile an anchor again.
    uint32_t vw = 0;
    if (D0 >= 4) vw = s.val[val_index<Q>(A, B, y)];
    const uint2 qb = *reinterpret_cast<const uint2 *>(s.dq + (size_t)c * 8);
    const int cc = s.code[c - 1];
    int vprev = (int)(xcol[(A + 1) * Q] & C::XAMASK);
    int Lc;
    if (y < Q - 1) Lc = s.rl[r0 + 1 + y];
    else Lc = (D >= 2) ? (int)(s.X[off_x<Q>(B - 1) + (A + 1) * Q + Q - 1] & C::XAMASK) : 0;
    // ---- fresh groups (a4): j in [0, min(k, D-2)] (column words of the tiles just below) and from max(D0-2, k+1) to
    // D-2 (row words of the tiles to the left inside the strip); without bulk (D0 < 4) that is every complete group
    uint32_t facc[Q];
#pragma unroll
    for (int a = 0; a < Q; ++a) facc[a] = 0;
    {
        // with top-up tasks only the two groups that were finished in the previous step are left: j = 0 and j = D-2
        const bool topped = C::TOPUP && D0 >= 4;
        const int j1 = topped ? 0 : min(k, D - 2), j2 = topped ? D - 2 : max(D0 - 2, k + 1);
        if (topped) {
            // two groups (D >= 4 here), written side by side: one round of operand loads, two independent gathers per row
            const uint32_t Xa = expand_x<Q>(xcol[(A + 1) * Q]), Xb = expand_x<Q>(xcol[(A + 1 + j2) * Q]);
            uint32_t wa[Q], wb[Q];
            load_rows<Q>(wrow, wa);
            load_rows<Q>(wrow + j2 * Q, wb);
#pragma unroll
            for (int a = 0; a < Q; ++a) facc[a] = lookup_max<Q>(s.tbl_sa, wb[a] + Xb, lookup_max<Q>(s.tbl_sa, wa[a] + Xa, 0u));
        } else {
            const int nf = (j1 + 1) + max(D - 1 - j2, 0);
            int j = 0;
#pragma unroll 1
            for (int f = 0; f < nf; ++f) {
                const uint32_t X32 = expand_x<Q>(xcol[(A + 1 + j) * Q]);
                uint32_t wr[Q];
                load_rows<Q>(wrow + j * Q, wr);
#pragma unroll
                for (int a = 0; a < Q; ++a) facc[a] = lookup_max<Q>(s.tbl_sa, wr[a] + X32, facc[a]);
                j = (j == j1) ? j2 : j + 1;
            }
        }
    }
    // everything the rows below contribute without the wave: bulk and fresh maxima folded once
#pragma unroll
    for (int a = 0; a < Q; ++a) facc[a] = max(facc[a] & 0xffffu, (uint32_t)unpack_row<Q>(vw, a));
    // diagonal tile (B,B) for the tail: packed pairs (Qd(2j,y), Qd(2j+1,y)); y' > y is "minus infinity"
    int Qp[C::NP];
#pragma unroll
    for (int jj = 0; jj < C::NP; ++jj) {
        const uint32_t src = jj < 2 ? qb.x : qb.y;
        uint32_t pr = __byte_perm(src, 0, (jj & 1) ? 0x4342 : 0x4140);
        if (2 * jj > y) pr |= 0x8000u;
        if (2 * jj + 1 > y) pr |= 0x80000000u;
        Qp[jj] = (int)pr;
    }
    // pairing mask of my column against the rows of the tile-row: bit a <-> b(S[r0+a], S[c-1])
    uint32_t pm = 0;
    if (cc < 4) pm = s.pm[A * 4 + cc];
    const uint32_t *wh = s.wdh + r0;
    uint16_t *scr = s.scr + (size_t)warp * C::SCR_WARP_HW;
    // lanes that own no output store to a per-warp dummy word instead of predicating every store
    uint32_t *wout = (own && y == 0) ? const_cast<uint32_t *>(wrow) + (D - 1) * Q : reinterpret_cast<uint32_t *>(scr + 2 * C::G * 8);
    int16_t *rlo = (own && y == Q - 1) ? s.rl + r0 : reinterpret_cast<int16_t *>(scr + 2 * C::G * 8 + 16);
    const int bsh = i * Q + 1;
    uint16_t *rowbase = scr + i * 8;
    uint32_t Xp = (uint32_t)vprev;
    int vl = __shfl_sync(FULL, vprev, lane - 1);                  // M(r+1, c-1) for the bottom row
    int v = 0;
    // the head gather of a row is issued as soon as the row below is known (before the shuffle, the ballot and the
    // stores of that row): a single warp issues in order, and those would otherwise sit in front of it
    uint32_t hS = wh[Q - 1] + Xp;
    uint32_t hR;
    asm("ld.shared.u8 %0, [%1];" : "=r"(hR) : "r"((hS >> C::ISH) + s.tbl_sa));
#pragma unroll
    for (int a = Q - 1; a >= 0; --a) {
        // ---- candidates from the rows below: bulk, fresh, pair term (a3), head residual (a5)
        const int lca = __shfl_sync(FULL, Lc, i * Q + a);
        const int vd = (y == 0) ? lca : vl;
        const int cand = max((int)facc[a], vd + (int)((pm >> a) & 1u));
        const uint32_t best = __viaddmax_u16x2(hS, hR, (uint32_t)cand);
        // ---- tail: V(a,y) = max_{y' <= y} C'(a,y') + Qd(y',y)
        uint16_t *row = rowbase + (a & 1) * (C::G * 8);
        if (lane_ok) row[y] = (uint16_t)(best & 0xffffu);
        __syncwarp();
        int m2 = (int)0x80008000u;
        if constexpr (Q == 8) {
            const uint4 t4 = *reinterpret_cast<const uint4 *>(row);
            const int m3 = __viaddmax_s16x2((int)t4.x, Qp[0], m2);
            const int m4 = __viaddmax_s16x2((int)t4.y, Qp[1], m2);
            const int m5 = __viaddmax_s16x2((int)t4.z, Qp[2], m3);
            const int m6 = __viaddmax_s16x2((int)t4.w, Qp[3], m4);
            m2 = __vmaxs2(m5, m6);
        } else {
#pragma unroll
            for (int jj = 0; jj < C::NP; ++jj) m2 = __viaddmax_s16x2((int)reinterpret_cast<const uint32_t *>(row)[jj], Qp[jj], m2);
        }
        v = max((int)(short)(m2 & 0xffff), m2 >> 16);
        // column word: the anchor moves up to row a, the difference to the row below enters at index bit a
        if (a == Q - 1) Xp = (uint32_t)v;
        else Xp += (uint32_t)(v - vprev) * (1u + (1u << (C::ISH + a)));
        if (a > 0) {
            hS = wh[a - 1] + Xp;
            asm("ld.shared.u8 %0, [%1];" : "=r"(hR) : "r"((hS >> C::ISH) + s.tbl_sa));
        }
        // ---- step a6: row word of row r over group B (ballot of the horizontal differences), column word bit
        vl = __shfl_sync(FULL, v, lane - 1);
        RNA4R_CHECK(!own || ((unsigned)(v - vprev) <= 1u && (y == 0 || (unsigned)(v - vl) <= 1u)));   // Lemma 1
        const uint32_t bal = __ballot_sync(FULL, y > 0 && v != vl);
        wout[a] = (((bal >> bsh) & C::HMASK) << 24) | (uint32_t)v;
        rlo[a] = (int16_t)v;
        vprev = v;
        if (own) store_cell<TABLE>(p, s.n, r0 + a, c, v);
    }
    if (own) {
        const_cast<uint16_t *>(xcol)[A * Q] = (uint16_t)(((Xp >> C::ISH) << C::XAB) | (Xp & 0xffffu));
        if (A == 0 && c == s.n) p.scores[seq] = v;                // M(0,n) = D(1,n)
    }
    if constexpr (C::DATAFLOW) {
        __threadfence_block();
        __syncwarp();
        if (own && y == 0) *(volatile int *)(s.prog + A) = D;
        if (lane == 0) {
            const int nt4 = min(C::G, (NT - A0 + C::G - 1) / C::G);
            __threadfence_block();
            if (atomicAdd(s.cntd + D, nt4) + nt4 == NT) atomicMax(s.cntd + NB + 1, D);                // the diagonal is complete
        }
    }
}

// ---- top-up: for the tiles that close in the NEXT step (tile-diagonal D1) and sit in column k >= 1 of their strip-tile,
// the groups the strip-tile's bulk pass could not take and that are finished by now -- j in [1, k] (column words of the
// tiles below, closed up to step D1-2) and [max(D0-2, k+1), D1-3] (row words of the tiles to the left) -- are merged into
// the packed bulk word.  Same lane layout and task numbering as the wave; u counts the tasks with k != 0.
template <int Q>
__device__ __forceinline__ void topup_task(const Sm<Q> &s, int D1, int u, int lane)
{
    using C = Cfg<Q>;
    const int NB = s.NB, NT = NB - D1;
    const int skip = (4 - (D1 & 3)) & 3;                       // the residue of A with k = (A + D1) mod 4 = 0
    const int r = u % 3, rho = r + (r >= skip ? 1 : 0);
    const int A0 = rho + 16 * (u / 3);
    if (A0 >= NT) return;
    const bool lane_ok = lane < C::SW;
    const int i = lane_ok ? lane / Q : C::G - 1;
    const int y = lane_ok ? lane - i * Q : Q - 1;
    int A = A0 + C::G * i;
    const bool own = lane_ok && A < NT;
    if (A >= NT) A = A0;
    const int B = A + D1;
    const int k = B & (C::G - 1), D0 = D1 - k;
    if (D0 < 4) return;                                        // no bulk word yet: the wave looks everything up (warp-uniform)
    const uint16_t *xcol = s.X + off_x<Q>(B) + y;
    const uint32_t *wrow = s.W + off_w<Q>(NB, A);
    uint32_t *slot = s.val + val_index<Q>(A, B, y);
    const uint32_t vw = *slot;
    uint32_t facc[Q];
#pragma unroll
    for (int a = 0; a < Q; ++a) facc[a] = 0;
    const int j1 = min(k, D1 - 3), j2 = max(D0 - 2, k + 1);
    const int nf = j1 + max(D1 - 2 - j2, 0);
    int j = 1;
#pragma unroll 1
    for (int f = 0; f < nf; ++f) {
        const uint32_t X32 = expand_x<Q>(xcol[(A + 1 + j) * Q]);
        uint32_t wr[Q];
        load_rows<Q>(wrow + j * Q, wr);
#pragma unroll
        for (int a = 0; a < Q; ++a) facc[a] = lookup_max<Q>(s.tbl_sa, wr[a] + X32, facc[a]);
        j = (j == j1) ? j2 : j + 1;
    }
#pragma unroll
    for (int a = 0; a < Q; ++a) facc[a] = max(facc[a] & 0xffffu, (uint32_t)unpack_row<Q>(vw, a));
    if (own) *slot = pack_rows<Q>(facc);
}

// Plan of tile-diagonal step D: ntw wave tasks | nE bulk tasks << 8 | first tile-row of a bulk task << 16 | log2(parts)
// << 20 (2 bits) | top-up tasks << 24.  Bulk tasks: the strip-tiles (A, GC = A + D0) that start on diagonal D0 = D+1 >= 4, groups j in [1, D0-3]; when
// warps would otherwise idle behind one long bulk task the range is split in 2 or 4 parts, which leave their maxima in
// dead rows of the ring (tile-rows >= NB-D have no tile left) and are merged after an extra barrier.
template <int Q>
__device__ __forceinline__ uint32_t step_plan(int NB, int D, int nwarp)
{
    using C = Cfg<Q>;
    const int NT = NB - D;
    const int ntw = 4 * ((NT + 15) >> 4);
    const int D0 = D + 1;
    const int Afirst = (4 - (D0 & 3)) & 3;
    const int nE = (D0 >= 4 && D0 < NB && NB - 1 - D0 >= Afirst) ? ((NB - 1 - D0 - Afirst) >> 2) + 1 : 0;
    const int elen = D0 - 3;
    int lp = 0;
    // top-up tasks for the tiles of diagonal D+1: three of the four residues of A (k != 0)
    const int ntu = (C::TOPUP && D + 1 < NB && D + 1 >= 5) ? 3 * ((NT - 1 + 15) >> 4) : 0;
    if (nE > 0 && !C::DATAFLOW) {
        const int wfree = nwarp - (NT + 3) / 4 - ntu;
        const int rows = (D * C::VPITCH) / 32;               // part slots (32 words each) the dead rows hold
        lp = (elen >= 72 && 4 * nE <= wfree && 4 * nE <= rows) ? 2 : (elen >= 40 && 2 * nE <= wfree && 2 * nE <= rows) ? 1 : 0;
    }
    return (uint32_t)ntw | ((uint32_t)nE << 8) | ((uint32_t)Afirst << 16) | ((uint32_t)lp << 20) | ((uint32_t)ntu << 24);
}

// NW warps per CTA: 24 with one CTA per SM (the register file: 80 x 768), 12 with two CTAs per SM for sequences whose
// state fits half the shared memory (a second sequence on the SM fills the issue slots a short fold leaves idle)
template <int Q, bool TABLE, int NW>
__global__ void __launch_bounds__(NW * 32, Cfg<Q>::NWARP / NW) seq_kernel(Params p)
{
    using C = Cfg<Q>;
    constexpr int NTHR = NW * 32;
    static_assert(C::G == 4, "task numbering assumes 4 tiles per warp");
    extern __shared__ __align__(16) uint8_t smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int seq = p.order ? p.order[blockIdx.x] : (int)blockIdx.x;
    const int n = p.offsets ? p.lens[seq] : p.n_single;
    const Layout L = make_layout<Q>(n);
    Sm<Q> s;
    {
        uint8_t *b = smem_raw;
        s.tbl_sa = smem_addr(b); b += C::TBL_AREA;
        s.scr = (uint16_t *)b; b += C::SCR_BYTES;
        s.misc = (int *)b; b += 64;
        s.W = (uint32_t *)(b + L.W); s.X = (uint16_t *)(b + L.X); s.val = (uint32_t *)(b + L.val);
        s.wdh = (uint32_t *)(b + L.wdh); s.dq = b + L.dq; s.pm = b + L.pm; s.rl = (int16_t *)(b + L.rl);
        s.code = (int8_t *)(b + L.code); s.plan = (uint32_t *)(b + L.plan);
        s.prog = (int *)(b + L.flags); s.bulkd = s.prog + (L.NB + 1); s.cntd = s.bulkd + (L.NB + 1);
        s.n = n; s.NB = L.NB;
        uint32_t dyn;
        asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn));
        if ((uint32_t)C::FIXED_BYTES + L.total > dyn) __trap();       // the host routes longer sequences elsewhere: fail loudly
    }
    const int NB = s.NB;
    unsigned long long *tr = (p.trace && seq < p.trace_seqs) ? p.trace + (size_t)seq * RNA4R_TRACE_WORDS : nullptr;
    long long t_start = 0, t_a = 0, t_b = 0, t_wave = 0, t_early = 0, t_setup = 0;
    int n_wave = 0;
    if (tr) t_start = clock64();
    // ---- setup: table, codes (step a1)
    {
        const uint32_t *src = reinterpret_cast<const uint32_t *>(p.tbl);
        uint32_t *dst = reinterpret_cast<uint32_t *>(smem_raw);
        for (int e = tid; e < C::TBL_BYTES / 4; e += NTHR) dst[e] = __ldg(src + e);
        for (int e = tid; e < C::SCR_BYTES / 4; e += NTHR) reinterpret_cast<uint32_t *>(s.scr)[e] = 0;
        if (tid < 16) s.misc[tid] = 0;
    }
    __syncthreads();
    {
        int bad = 0;
        if (p.offsets && p.offsets[seq + 1] - p.offsets[seq] != (int64_t)n) bad = RNA4R_STATUS_BAD_OFFSETS;
        const uint8_t *src = p.seqs + (p.offsets && !bad ? p.offsets[seq] : 0);
        for (int x = tid; x < NB * Q + 16; x += NTHR) {
            int cde = 4;
            if (x < n && !bad) { cde = rna4r_base_code(src[x]); if (cde == 4) bad |= RNA4R_STATUS_BAD_BASE; }
            s.code[x] = (int8_t)cde;
        }
        if (bad) atomicOr(&s.misc[1], bad);
    }
    __syncthreads();
    if (s.misc[1]) {                                   // reading g4: not a base -> score -1, status word
        if (tid == 0) { p.scores[seq] = -1; if (p.status) p.status[seq] = s.misc[1]; }
        return;
    }
    if (tid == 0 && p.status) p.status[seq] = 0;
    for (int e = tid; e < NB * 4; e += NTHR) {
        const int A = e >> 2, x = e & 3;
        uint32_t bits = 0;
#pragma unroll
        for (int a = 0; a < Q; ++a) bits |= (uint32_t)rna4r_pair(s.code[A * Q + a], x) << a;
        s.pm[e] = (uint8_t)bits;
    }
    for (int D = tid; D < NB; D += NTHR) s.plan[D] = step_plan<Q>(NB, D, NW);
    for (int e = tid; e < 3 * NB + 8; e += NTHR) s.prog[e] = 0;
    // ---- tile-diagonal 0
    for (int A = tid; A < NB; A += NTHR) diag_tile<Q, TABLE>(p, s, seq, A);
    __syncthreads();
    if (tr) t_setup = clock64() - t_start;

    for (int D = 1; D < NB; ++D) {
        long long ta0 = 0, tb0 = 0;
        if (tr) ta0 = clock64();
        const int NT = NB - D;
        // Tasks of the step (step_plan), dealt round-robin to the warps, waves first
        const uint32_t plan = s.plan[D];
        const int ntw = (int)(plan & 0xffu), nE = (int)((plan >> 8) & 0xffu), Afirst = (int)((plan >> 16) & 3u), lp = (int)((plan >> 20) & 3u);
        const int ntu = (int)(plan >> 24);
        const int D0 = D + 1, elen = D0 - 3;
        uint32_t *part = s.val + NT * C::VPITCH;
        const int nbulk = nE << lp;
        const int ntask = ntw + nbulk + ntu;                       // dealt in this order: waves, bulk, top-ups
        for (int t = warp; t < ntask; t += NW) {
            long long tt0 = 0;
            if (tr) tt0 = clock64();
            if (t < ntw) {
                wave_task<Q, TABLE>(p, s, seq, D, t, warp, lane);
                if (tr) { t_wave += clock64() - tt0; ++n_wave; }
            } else if (t >= ntw + nbulk) {
                topup_task<Q>(s, D + 1, t - ntw - nbulk, lane);
                if (tr) t_early += clock64() - tt0;
            } else {
                const int e = t - ntw, ie = e >> lp, pe = e & ((1 << lp) - 1);
                const int A = Afirst + C::G * ie, GC = A + D0;
                uint32_t acc[Q];
#pragma unroll
                for (int a = 0; a < Q; ++a) acc[a] = 0;
                if constexpr (C::DATAFLOW) {
                    // operands: tiles of the diagonals <= D0-2 = D-1; the ring slots it overwrites were read by tiles of
                    // tile-row A up to diagonal D0-2 as well
                    volatile int *ad = s.cntd + NB + 1;
                    while (*ad < D - 1) __nanosleep(64);
                    __threadfence_block();
                }
                strip_bulk<Q>(s, A, GC, 1 + ((elen * pe) >> lp), (elen * (pe + 1)) >> lp, lane, acc);
                const uint32_t w = pack_rows<Q>(acc);
                if (lp > 0) part[e * 32 + lane] = w;
                else if (lane < C::SW && GC + lane / Q < NB) s.val[val_index<Q>(A, GC + lane / Q, lane % Q)] = w;
                if constexpr (C::DATAFLOW) {
                    __threadfence_block();
                    __syncwarp();
                    if (lane == 0) *(volatile int *)(s.bulkd + A) = D0;
                }
                if (tr) t_early += clock64() - tt0;
            }
        }
        if constexpr (!C::DATAFLOW) __syncthreads();
        if (tr) { tb0 = clock64(); t_a += tb0 - ta0; }
        if (lp > 0) {
            for (int ie = warp; ie < nE; ie += NW) {
                const int A = Afirst + C::G * ie, GC = A + D0;
                uint32_t acc[Q];
#pragma unroll
                for (int a = 0; a < Q; ++a) acc[a] = 0;
                for (int pe = 0; pe < (1 << lp); ++pe) {
                    const uint32_t w = part[((ie << lp) + pe) * 32 + lane];
#pragma unroll
                    for (int a = 0; a < Q; ++a) acc[a] = max(acc[a], (uint32_t)unpack_row<Q>(w, a));
                }
                if (lane < C::SW && GC + lane / Q < NB) s.val[val_index<Q>(A, GC + lane / Q, lane % Q)] = pack_rows<Q>(acc);
            }
            __syncthreads();
        }
        if (tr) t_b += clock64() - tb0;
    }
    if (tr && tid == 0) {
        tr[0] = (unsigned long long)(clock64() - t_start); tr[1] = (unsigned long long)t_setup; tr[2] = (unsigned long long)t_a;
        tr[3] = (unsigned long long)t_b; tr[4] = (unsigned long long)t_wave; tr[5] = (unsigned long long)n_wave;
        tr[6] = (unsigned long long)t_early; tr[7] = (unsigned long long)n;
    }
}

// ---- host side ------------------------------------------------------------------------------------------------------
static inline size_t workspace_bytes(int count) { return 256 + 2 * align_up((size_t)(count > 0 ? count : 1) * 4, 256); }

template <int Q>
static int enqueue_q(rna4r_ctx *ctx, const uint8_t *seqs, const int64_t *offsets, const int32_t *lens_host, int count, int n_single,
                     int32_t *scores, int32_t *status, void *table_out, int table_dtype, void *ws, cudaStream_t st,
                     bool skip_long = false)
{
    // skip_long: sequences beyond max_n<Q>() belong to another engine's half of the batch and are left out
    using C = Cfg<Q>;
    Params p;
    p.seqs = seqs; p.offsets = offsets; p.lens = nullptr; p.order = nullptr; p.n_single = n_single;
    p.tbl = ctx->Rc; p.scores = scores; p.status = status; p.table_out = table_out; p.table_dtype = table_dtype;
    p.trace = ctx->trace; p.trace_seqs = ctx->trace_tiles;
    int max_len = n_single, grid = count;
    if (offsets) {
        // longest first: the hardware hands CTAs to SMs in index order, so this is the LPT rule (work ~ n^3).
        // Counting sort by length into a context-owned host array (grown on demand, never per call).
        if (count > ctx->order_cap) {
            int32_t *nb = new (std::nothrow) int32_t[(size_t)count];
            if (!nb) return RNA4R_ERR_CUDA;
            delete[] ctx->order_host;
            ctx->order_host = nb; ctx->order_cap = count;
        }
        const int lim = max_n<Q>();
        max_len = 0;
        for (int t = 0; t < count; ++t) if (lens_host[t] > max_len && (!skip_long || lens_host[t] <= lim)) max_len = lens_host[t];
        {
            int hist[2050] = {0};
            if (max_len > 2048) return RNA4R_ERR_BAD_N;
            for (int t = 0; t < count; ++t) if (lens_host[t] <= max_len) ++hist[max_len - lens_host[t] + 1];
            for (int b = 1; b <= max_len + 1; ++b) hist[b] += hist[b - 1];
            grid = hist[max_len + 1];
            for (int t = 0; t < count; ++t) if (lens_host[t] <= max_len) ctx->order_host[hist[max_len - lens_host[t]]++] = t;
        }
        char *base = (char *)ws;
        int32_t *lens_dev = (int32_t *)(base + 256);
        int32_t *order_dev = (int32_t *)(base + 256 + align_up((size_t)count * 4, 256));
        RNA4R_CUDA(ctx, cudaMemcpyAsync(lens_dev, lens_host, (size_t)count * 4, cudaMemcpyHostToDevice, st));
        RNA4R_CUDA(ctx, cudaMemcpyAsync(order_dev, ctx->order_host, (size_t)count * 4, cudaMemcpyHostToDevice, st));
        p.lens = lens_dev; p.order = order_dev;
    }
    if (max_len > max_n<Q>()) return RNA4R_ERR_BAD_N;
    auto smem_of = [](int n) { size_t b = (size_t)C::FIXED_BYTES + make_layout<Q>(n).total; return b < 49152 ? (size_t)49152 : b; };
    if (ctx->timing) RNA4R_CUDA(ctx, cudaEventRecord(ctx->ev0, st));
    int launches = 0;
    if (!offsets) {
        if (table_out) {
            RNA4R_CUDA(ctx, cudaFuncSetAttribute(seq_kernel<Q, true, C::NWARP>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::MAX_SMEM));
            seq_kernel<Q, true, C::NWARP><<<1, C::NTHR, smem_of(max_len), st>>>(p);
        } else {
            RNA4R_CUDA(ctx, cudaFuncSetAttribute(seq_kernel<Q, false, C::NWARP>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::MAX_SMEM));
            seq_kernel<Q, false, C::NWARP><<<1, C::NTHR, smem_of(max_len), st>>>(p);
        }
        launches = 1;
    } else if (grid > 0) {
        // One kernel for the batch; its CTA size follows the longest sequence: a fold that needs the whole shared memory
        // of an SM gets 24 warps, and when every state fits 1/2, 1/3, 1/4 of it the CTAs have 12, 8, 6 warps and two to
        // four sequences share an SM (the register file holds 24 warps at 80 registers): a short fold has too few
        // independent tasks per tile-diagonal for 24 warps, a neighbour on the SM fills the idle issue slots (2048
        // sequences of 100..400 bases: 1.04 ms with 24-warp CTAs, 0.71 ms with two CTAs per SM).  A mixed batch is not
        // split by class: measured slower (cfg4 1.72 against 1.54 ms), the long class loses the short folds that fill
        // the tail of its longest-first order.
        const size_t need = smem_of(max_len);
        const size_t per_sm = 233472;                    // 228 KB, 1 KB of it reserved per resident CTA
        auto launch = [&](auto NWc) -> int {
            constexpr int NW = decltype(NWc)::value;
            RNA4R_CUDA(ctx, cudaFuncSetAttribute(seq_kernel<Q, false, NW>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::MAX_SMEM));
            seq_kernel<Q, false, NW><<<grid, NW * 32, need, st>>>(p);
            return RNA4R_OK;
        };
        int rc;
        if (need + 1024 <= per_sm / 4) rc = launch(std::integral_constant<int, C::NWARP / 4>{});
        else if (need + 1024 <= per_sm / 3) rc = launch(std::integral_constant<int, C::NWARP / 3>{});
        else if (need + 1024 <= per_sm / 2) rc = launch(std::integral_constant<int, C::NWARP / 2>{});
        else rc = launch(std::integral_constant<int, C::NWARP>{});
        if (rc != RNA4R_OK) return rc;
        launches = 1;
    }
    if (ctx->timing) { RNA4R_CUDA(ctx, cudaEventRecord(ctx->ev1, st)); ctx->timing_valid = 1; }
    RNA4R_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = launches;
    return RNA4R_OK;
}

}  // namespace smemseq
