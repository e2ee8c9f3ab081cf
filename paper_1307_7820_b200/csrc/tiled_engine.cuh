// tiled_engine.cuh -- RNA4R_ENGINE_TILED: the B200 design of the two-vector Four-Russians fill.
//
// Coordinates.  The paper's D(i,j) (1-based) is held as a matrix M(r,c) = D(r+1, c),
// r,c in [0,n]: M(r,c) = 0 for c <= r+1, and eq. (1) becomes a pure max-plus closure
//     M(r,c) = max{ b(S[r],S[c-1]) + M(r+1,c-1),  max_{r<t<c} M(r,t) + M(t,c) }.
// With this shift the paper's two offset groupings (columns (0..q-1),(q..2q-1),.. and rows
// (1..q),(q+1..2q),..) are the SAME grouping of the split index t: group g is
// t in [gq, gq+q).
//
// Two-vector step (eq. (3)).  For group g, row r, column c:
//     max_{t in g} M(r,t)+M(t,c) = M(r,gq) + M(gq,c) + Rc[h][v]
//   h = the q-1 horizontal difference bits of M(r,gq..gq+q-1)  (v_1..v_{q-1};  v_0 = 0)
//   v = the q-1 vertical   difference bits of M(gq..gq+q-1,c)  (|vbar_1|..|vbar_{q-1}|; vbar_0 = 0)
// Each (row, group) is one 32-bit word W = anchor M(r,gq) + index bits h, and each (group, column) one word
// X = anchor M(gq,c) + index bits v  (HB = q-1 bits each, SH = 2*HB index bits, h above v).  Then S = W + X
// carries the table index and the anchor sum in disjoint fields, and the candidate is S + Rc[idx] on the value
// field.  The value sits in the low halfword and the index in the high one (binary for q <= 9, ternary above), so
// that the gather address is (S >> 16) + base (one LEA.HI) and "max(acc, S + rv)" is one DPX instruction
// (VIADDMNMX.U16x2) -- add, address, LDS.U8, add-max.  The index bits left in a candidate are harmless: they never
// change the order of the value field.  q >= 10 indexes a table of 3^(q-1) entries in base 3 (Cfg::TERN).
//
// Decomposition.  Super-tiles of T = 8q cells (8 groups) per side.  For super-tile (I,J), I < J:
//   * every group lying in a block K strictly between I and J is a "full group" for ALL T*T cells
//     (Alg. 1 lines 15-19): a max-plus product of the row panel of (I,K) with the
//     column panel of (K,J) through Rc -- the bulk, no dependency inside the tile;
//   * groups inside blocks I and J depend on cells of (I,J) itself: the closure, a 2T-1 step
//     anti-diagonal wavefront inside the CTA.  The paper's residual loops
//      are done as MASKED lookups: a partial group is a lookup whose not
//     yet known difference bits are zero (DESIGN.md section 4.3 proves this is exact).
// Work units (tasks) are listed step by step (step = super-tile diagonal J-I), claimed in order from
// one atomic counter by a persistent grid, and ordered by acquire/release flags instead of a grid
// barrier per diagonal ("Synchronize with other processes").
#pragma once
#include "common.cuh"

#ifndef RNA4R_TERN_MIN_Q
#define RNA4R_TERN_MIN_Q 9        // smallest q that indexes the table in base 3 (Cfg::TERN)
#endif

namespace tiled {



template <int Q>
struct Cfg {
    static constexpr int T = 8 * Q;            // cells per super-tile side
    static constexpr int HB = Q - 1;           // informative bits per vector
    static constexpr int SH = 2 * HB;          // table index bits
    static constexpr uint32_t IDXMASK = (1u << SH) - 1u;
    // Word format (F16, every q): value in bits [0,16), table index in bits [16,32): a candidate is
    // max(acc, S + rv) on the low halfword -- ONE DPX instruction (VIADDMNMX.U16x2; the high halfword carries
    // harmless index bits), and the gather address is (S >> 16) + base -- one LEA.HI.
    //
    // q <= 8: BINARY index h * pitch + v.  The table rows (2^HB bytes, one per h) are stored with a
    // pitch of 2^HB + 4 bytes.  A row of 128 bytes covers the 32 banks exactly once, so with the natural
    // pitch the bank of a gather depends on v alone and the closure's gathers -- different h per lane, partial (mostly
    // zero) v -- pile up on a few banks (ncu: 7-way conflicts).  With the padded pitch the bank is (h + v/4) mod 32; the
    // bulk product (one h per warp) stays conflict-free.  The index field of a row word is then h * TBL_PITCH (a sum
    // of per-bit constants), not a bit field; the column word still adds v.
    //
    // q >= 9 (RNA4R_TERN_MIN_Q): TERNARY index.  The black box sees the two vectors only through d_k = v_k - |vbar_k| in
    // {-1,0,1}: R[h][v] = max(0, max_k sum_{k'<=k} d_k').  A table indexed by sum_k (h_k + 1 - v_k) 3^k has 3^(q-1)
    // entries (6 561 bytes at q = 9, 19 683 at q = 10, 59 049 at q = 11, against 2^16, 2^18 and 2^20), and the index is still the sum of a
    // row part sum h_k 3^k and a column part sum (1 - v_k) 3^k -- base-3 digits 0..2, no carries -- so S = W + X and
    // the four-instruction lookup stay as they are.  The price: the gathers of a warp scatter over the whole table
    // (bank conflicts, as a binary table wider than 128 bytes per row has them too), where the layout of q <= 8 has
    // none in the bulk product.  Measured on cfg5 (n = 16384): q = 9 37.3 -> 27.1 ms, q = 10 (nibble-packed binary
    // table before) 41.7 -> 23.6 ms, q = 11 25.5 ms (not possible before).
    static constexpr bool TERN = (Q >= RNA4R_TERN_MIN_Q);
    static constexpr bool F16 = true;
    static constexpr int VSHIFT = 0;           // position of the value field
    static constexpr int ISHIFT = 16;          // position of the index field
    __host__ __device__ static constexpr uint32_t pow3(int k) { return k <= 0 ? 1u : 3u * pow3(k - 1); }
    static constexpr uint32_t TERN_C0 = (pow3(HB) - 1u) / 2u;      // index part of a column word without set bits: sum_k 3^k
    static_assert(TERN ? pow3(HB) <= 65536u : SH <= 16, "the table index has to fit the high halfword");
    static constexpr int TBL_PITCH = TERN ? 1 : (Q <= 8 ? (1 << HB) + 4 : (1 << HB));     // q = 9: 256 x 260 would overflow the halfword
    static constexpr int TBL_BYTES = TERN ? (int)pow3(HB) : (1 << HB) * TBL_PITCH;
    static constexpr uint32_t VMASK = ((1u << HB) - 1u) << ISHIFT;      // the v bits of a (binary) column word
    static constexpr int TBL_AREA = (TBL_BYTES + 15) / 16 * 16;
    static constexpr int PTHR = 4 * T;         // threads that take part in a bulk product (T columns x 4 row blocks)
    static constexpr int WTHR = PTHR > 256 ? PTHR : 256;   // product threads, and at least the 8 closure warps
    static constexpr int NTHR = WTHR + 128;    // + 4 warps: a closure needs NROLE = NWV + NMH + 8 warps
    static constexpr int MIN_CTAS = (Q <= 8) ? 3 : ((TERN && Q <= 10) ? 2 : 1);   // register budget: 3 CTAs per SM with the byte table of q <= 8,
                                               // 2 with the ternary tables of q = 9, 10 (q = 9 at 3 CTAs: 48 registers, spills, 3 % faster on cfg5 -- not taken)
    static constexpr int RPT = Q;              // product phase: a thread owns RPT rows x 2 columns (c and c + T/2): the warp-uniform
    static constexpr int HT = T / 2;           // row words are loaded once for 2*RPT lookups (a broadcast LDS.128 costs 2 wavefronts)
    static constexpr int TP = T + 8;           // pitch of the per-group word arrays (bank spread)
    static constexpr int VP = T + 10;          // pitch of the value arrays (int16) = 4q+5 words, odd and >= q/2 away from a multiple of 32:
                                               // a column (lanes = rows), a q-tile patch (4 rows x q columns) and a skewed wavefront step
                                               // (lane y on row a+y, column c+y) are all bank-conflict-free
    static constexpr int PANEL_WORDS = 8 * T;  // words in one row or column panel
    static constexpr int REC_BYTES = 2 * PANEL_WORDS * 4 + 2 * T * 2;   // PH, PV, top row, right column
    static constexpr int WROWS = 16;           // word-array rows: 8 groups of block I, 8 of block J
    // shared-memory layout: [tbl | guard | Wst | Xst | val (guard rows around) | val2 | val3 | stg | codeR | codeC | misc | mbar]
    // The unrolled closure steps address val and Wst with immediate offsets; lanes outside their window
    // read up to Q rows beyond either end of the arrays (values ignored): the guards keep those reads inside.
    static constexpr int W_GUARD = 64;         // bytes before Wst
    static constexpr int W_BYTES = WROWS * TP * 4;
    static constexpr int PRE_BYTES = (W_GUARD + 2 * W_BYTES + 15) / 16 * 16;
    static constexpr int VAL_ROWS = T + 1 + 2 * Q;   // Q guard rows, rows 0..T, Q guard rows
    static constexpr int VAL_BYTES = ((VAL_ROWS * VP + 2) * 2 + 15) / 16 * 16;
    static constexpr int NSTG = 2;             // depth of the bulk product's operand ring
    static constexpr int STG_BYTES = NSTG * 2 * PANEL_WORDS * 4;
    static constexpr int VP2 = VP;             // pitch of val2 / val3
    static constexpr int VAL2_BYTES = (T * VP2 * 2 + 15) / 16 * 16;   // late products of block I+1 (kept apart: two warps merge concurrently)
    // closure warps: a warp runs G q-tiles of one anti-diagonal side by side (Q lanes each); NWV such warps cover
    // the <= 8 q-tiles of a macro-step; NMH helper warps prepare the next macro-step's older complete groups
    static constexpr int G = (32 / Q < 4) ? 32 / Q : 4;
    static constexpr int NWV = (8 + G - 1) / G;
    static constexpr int NMH = 2;
    static constexpr int NROLE = NWV + NMH + 8;          // + row/column loader, row/column publisher, 2 row-late, 2 column-late
    static constexpr int STEP_THREADS = (NWV + NMH) * 32;   // participants of the per-macro-step named barrier
    // mbarriers (each completes once per closure): [0,15) macro-step u done; [16,24) rows of q-row A of the left
    // tile loaded; [24,32) columns of q-column B of the tile below loaded; [32,47) everything macro-step u needs
    // from the late-product helpers has been merged: the left (right) half of q-row A's late products arrives at
    // u = 7-A (11-A), the lower (upper) half of q-column B's at u = B (B+4) -- see stepin_count()
    static constexpr int MB_STEP = 0, MB_ROW = 16, MB_COL = 24, MB_STEPIN = 32, MB_COUNT = 48;
    static constexpr int MB_PROD = 48, MB_TOTAL = 56;    // bulk product ring: operands landed [48,48+NSTG), buffer free [52,52+NSTG)
    __host__ __device__ static constexpr int stepin_count(int u) { return (u <= 3) ? 2 : (u <= 7) ? 4 : (u <= 11) ? 2 : 0; }
    static constexpr int MBAR_BYTES = MB_TOTAL * 8;
    static_assert(NROLE * 32 <= NTHR, "closure roles must fit the CTA");
    static constexpr int POST_BYTES = VAL_BYTES + 2 * VAL2_BYTES + STG_BYTES + ((2 * T + 15) / 16 * 16) + 64 + MBAR_BYTES;
    // The table sits at the START of the dynamic window.  F16: the gather address is (S >> 16) + base with no
    // mask; an idle lane's don't-care S can index up to 65535, so the window is at least 64 KB + 16 long and the
    // stray read stays inside it (its value is ignored).
    static constexpr size_t LAYOUT_BYTES = (size_t)TBL_AREA + PRE_BYTES + POST_BYTES;
    static constexpr size_t SMEM_BYTES = (F16 && LAYOUT_BYTES < 65536 + 16) ? 65536 + 16 : LAYOUT_BYTES;
};

struct SeqInfo {
    int n;         // sequence length
    int nt;        // super-tiles per side = n / T + 1
    int sbase;     // index of this sequence's first super-tile record
    int cbase;     // offset of this sequence's codes
    int invalid;   // != 0 if a byte was not a base
    int pad[3];
};

// header of the plan area (zeroed by one memset at the start of every fold)
struct PlanHdr {
    int counter;    // task claim counter
    int total;      // number of tasks
    int ntiles;     // allocation cursor: super-tile records
    int ncodes;     // allocation cursor: code bytes
    int pad[4];
};

constexpr int TASK_CLOSE = 0;
constexpr int TASK_PROD = 1;

struct Params {
    const uint8_t *seqs;
    const int64_t *offsets;   // device [count+1], or NULL for a single sequence of length n_single
    const int32_t *lens_dev;  // device copy of lens_host [count] (batch only): the geometry always follows the host plan
    const int32_t *map;       // NULL, or device [count]: sequence t of this call is sequence map[t] of the caller's batch
                              // (offsets, scores, status are indexed through it: a batch split between two engines)
    int32_t *status;          // NULL, or device [count]: RNA4R_STATUS_* bits per sequence
    int n_single;
    int count;
    int max_nt;
    int delta;
    PlanHdr *hdr;
    int *stepC;       // [max_nt] closure tasks per step, then segment base
    int *stepP;       // [max_nt] product tasks per step, then segment base
    int *curC;        // [max_nt] fill cursors
    int *curP;
    SeqInfo *seqinfo; // [count]
    int *done;        // [tiles] 1 when the super-tile's panels are published
    int *accstage;    // [tiles] product stages merged into acc so far
    int *rowprog;     // [tiles] q-rows (from the bottom) whose row words and right-column values are published
    int *colprog;     // [tiles] q-columns (from the left) whose column words and top-row values are published
    int4 *tasks;      // {seq, I | J << 16, kind, stage}
    int8_t *codes;    // per sequence nt*T codes (4 = padding)
    uint8_t *recs;    // super-tile records
    int16_t *acc;     // [tiles][T*T] bulk partial maxima
    const uint8_t *tbl;   // compact table in global memory (byte or nibble form)
    int32_t *scores;
    void *table_out;
    int table_dtype;
    unsigned long long *trace;   // NULL, or [tiles][8] phase stamps (ns) of the CLOSE tasks
    int trace_tiles;
    int sm_count;                // SMs of the device (role rotation of co-resident CTAs)
};

__host__ __device__ inline int nstages(int dp, int delta)
{
    // product stages of a target on super-tile diagonal dp: stage s runs at step
    // dp-1-s*delta and covers member diagonals m in [max(hi-delta+1, ceil(dp/2)), hi], hi = dp-2-s*delta
    const int mmin = (dp + 1) / 2;
    if (dp - 2 < mmin) return 0;
    return (dp - 2 - mmin) / delta + 1;
}
__host__ __device__ inline int tri_index(int nt, int I, int J) { return I * nt - (I * (I - 1)) / 2 + (J - I); }

// ------------------------------------------------------------------------------------------------
// planning kernels (tiny): per-sequence geometry, per-step task counts, task list
// ------------------------------------------------------------------------------------------------
template <int Q>
__global__ void plan_seq_kernel(Params p)
{
    // block <-> sequence; threads <-> steps
    constexpr int T = Cfg<Q>::T;
    const int t = blockIdx.x;
    if (t >= p.count) return;
    // The geometry follows lens_host (copied to lens_dev), as the host-side workspace plan does; a sequence whose
    // device offsets disagree with it is folded as padding and reported (score -1, RNA4R_STATUS_BAD_OFFSETS).
    const int n = p.offsets ? p.lens_dev[t] : p.n_single;
    const int nt = n / T + 1;
    if (threadIdx.x == 0) {
        SeqInfo si;
        si.n = n; si.nt = nt; si.pad[0] = si.pad[1] = si.pad[2] = 0;
        const int o = p.map ? p.map[t] : t;
        si.invalid = (p.offsets && p.offsets[o + 1] - p.offsets[o] != (int64_t)n) ? RNA4R_STATUS_BAD_OFFSETS : 0;
        si.sbase = atomicAdd(&p.hdr->ntiles, nt * (nt + 1) / 2);
        si.cbase = atomicAdd(&p.hdr->ncodes, nt * T);
        p.seqinfo[t] = si;
    }
    for (int D = threadIdx.x; D < nt; D += blockDim.x) {
        atomicAdd(&p.stepC[D], nt - D);
        int np = 0;
        for (int s = 0;; ++s) {
            const int dp = D + 1 + s * p.delta;
            if (dp > nt - 1) break;
            if (s < nstages(dp, p.delta)) np += nt - dp;
        }
        if (np) atomicAdd(&p.stepP[D], np);
    }
}

__global__ void plan_scan_kernel(Params p)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    int base = 0;
    for (int D = 0; D < p.max_nt; ++D) {
        const int c = p.stepC[D], q = p.stepP[D];
        p.stepC[D] = base; p.curC[D] = base; base += c;
        p.stepP[D] = base; p.curP[D] = base; base += q;
    }
    p.hdr->total = base;
}

template <int Q>
__global__ void plan_fill_kernel(Params p)
{
    // block <-> (sequence t, step D)
    const int t = blockIdx.x / p.max_nt, D = blockIdx.x % p.max_nt;
    const SeqInfo si = p.seqinfo[t];
    const int nt = si.nt;
    if (D >= nt) return;
    __shared__ int s_slot;
    if (threadIdx.x == 0) s_slot = atomicAdd(&p.curC[D], nt - D);
    __syncthreads();
    for (int I = threadIdx.x; I < nt - D; I += blockDim.x)
        p.tasks[s_slot + I] = make_int4(t, I | ((I + D) << 16), TASK_CLOSE, 0);
    for (int s = 0;; ++s) {
        const int dp = D + 1 + s * p.delta;
        if (dp > nt - 1) break;
        if (s >= nstages(dp, p.delta)) continue;
        __syncthreads();
        if (threadIdx.x == 0) s_slot = atomicAdd(&p.curP[D], nt - dp);
        __syncthreads();
        for (int I = threadIdx.x; I < nt - dp; I += blockDim.x)
            p.tasks[s_slot + I] = make_int4(t, I | ((I + dp) << 16), TASK_PROD, s);
    }
}

// bases -> codes, padded with 4 up to nt*T; flags invalid bytes (reading g4)
template <int Q>
__global__ void encode_kernel(Params p)
{
    constexpr int T = Cfg<Q>::T;
    for (int t = blockIdx.y; t < p.count; t += gridDim.y) {
        const SeqInfo si = p.seqinfo[t];
        const int len = si.nt * T;
        const bool readable = !(si.invalid & RNA4R_STATUS_BAD_OFFSETS);      // never read through offsets that failed the check
        const uint8_t *src = p.seqs + (p.offsets && readable ? p.offsets[p.map ? p.map[t] : t] : 0);
        bool bad = false;
        for (int x = blockIdx.x * blockDim.x + threadIdx.x; x < len; x += gridDim.x * blockDim.x) {
            int c = 4;
            if (x < si.n && readable) { c = rna4r_base_code(src[x]); bad |= (c == 4); }
            p.codes[si.cbase + x] = (int8_t)c;
        }
        if (bad) atomicOr(&p.seqinfo[t].invalid, RNA4R_STATUS_BAD_BASE);
    }
}

// Single fold: the whole plan (geometry, per-step task counts, task list) and the encoding in ONE launch.  Block D owns
// step D: it sums the task counts of the earlier steps itself (a few hundred terms), writes the step's CLOSE and PROD
// tasks in the order of the batch path, and encodes the bases of super-tile D.
template <int Q>
__global__ void plan_single_kernel(Params p)
{
    constexpr int T = Cfg<Q>::T;
    const int n = p.n_single, nt = n / T + 1;
    const int D = blockIdx.x, tid = threadIdx.x;
    auto prods_of = [&](int d) {
        int np = 0;
        for (int s = 0;; ++s) {
            const int dp = d + 1 + s * p.delta;
            if (dp > nt - 1) break;
            if (s < nstages(dp, p.delta)) np += nt - dp;
        }
        return np;
    };
    __shared__ int red[128];
    int part = 0;
    for (int d = tid; d < D; d += blockDim.x) part += (nt - d) + prods_of(d);
    red[tid] = part;
    __syncthreads();
    for (int w = blockDim.x / 2; w > 0; w >>= 1) {
        if (tid < w) red[tid] += red[tid + w];
        __syncthreads();
    }
    const int baseC = red[0], baseP = baseC + (nt - D);
    for (int I = tid; I < nt - D; I += blockDim.x) p.tasks[baseC + I] = make_int4(0, I | ((I + D) << 16), TASK_CLOSE, 0);
    int slot = baseP;
    for (int s = 0;; ++s) {
        const int dp = D + 1 + s * p.delta;
        if (dp > nt - 1) break;
        if (s >= nstages(dp, p.delta)) continue;
        for (int I = tid; I < nt - dp; I += blockDim.x) p.tasks[slot + I] = make_int4(0, I | ((I + dp) << 16), TASK_PROD, s);
        slot += nt - dp;
    }
    if (tid == 0) {
        if (D == nt - 1) p.hdr->total = slot;
        if (D == 0) { SeqInfo *si = p.seqinfo; si->n = n; si->nt = nt; si->sbase = 0; si->cbase = 0; }   // invalid: zeroed, OR-ed below
    }
    bool bad = false;
    for (int x = D * T + tid; x < (D + 1) * T; x += blockDim.x) {
        int c = 4;
        if (x < n) { c = rna4r_base_code(p.seqs[x]); bad |= (c == 4); }
        p.codes[x] = (int8_t)c;
    }
    if (bad) atomicOr(&p.seqinfo[0].invalid, RNA4R_STATUS_BAD_BASE);
}

// ------------------------------------------------------------------------------------------------
// fill kernel
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <int Q>
struct Smem {
    using C = Cfg<Q>;
    uint32_t *Wst;       // [WROWS][TP] row words:    groups 0..7 of block I (static), 8..15 of block J (own)
    uint32_t *Xst;       // [WROWS][TP] column words: groups 0..7 of block I (own),    8..15 of block J (static)
    uint8_t *tbl;        // compact table Rc
    uint32_t tbl_sa;     // its shared-space address
    int16_t *valraw;     // start of the value array including its guard rows
    int16_t *val;        // [(T+1)][VP] values; column 0 = right column of (I,J-1), row T = top row of (I+1,J)
    int16_t *val2;       // [T][VP2] late products of block K = I+1 (written by the column-late helper, merged by the closure warps)
    int16_t *val3;       // [T][VP2] older complete groups of the closure (written by the mini helpers one macro-step ahead)
    uint32_t *stg;       // [2][2][PANEL_WORDS] product operands, double buffered: [buf][0]=PH, [buf][1]=PV
    int8_t *codeR;       // [T] codes of the rows
    int8_t *codeC;       // [T] codes of the columns
    int *misc;           // [16]
    uint64_t *mbar;      // [8][8] mbarrier of q-tile (A,B) at mbar[B*8+A]: completes once per closure
    bool ok;             // the layout fits the dynamic shared memory of this launch
    __device__ explicit Smem(uint8_t *base)
    {
        uint8_t *p = base;
        tbl = p; tbl_sa = smem_addr(base); p += C::TBL_AREA;
        p += C::W_GUARD;
        Wst = (uint32_t *)p; p += C::W_BYTES;
        Xst = (uint32_t *)p; p += C::W_BYTES;
        p = base + C::TBL_AREA + C::PRE_BYTES;
        valraw = (int16_t *)p; val = valraw + Q * C::VP; p += C::VAL_BYTES;     // val[0] = row 0; Q guard rows on either side
        val2 = (int16_t *)p; p += C::VAL2_BYTES;
        val3 = (int16_t *)p; p += C::VAL2_BYTES;
        stg = (uint32_t *)p; p += C::STG_BYTES;
        codeR = (int8_t *)p; p += C::T;
        codeC = (int8_t *)p; p += C::T;
        p = base + ((p - base) + 15) / 16 * 16;
        misc = (int *)p; p += 64;
        mbar = (uint64_t *)p; p += C::MBAR_BYTES;
        uint32_t dyn;
        asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn));
        ok = (uint32_t)(p - base) <= dyn && dyn >= (uint32_t)C::SMEM_BYTES;
    }
};

// One table gather (the unit of work of this path): rv = Rc[index field of S].  SAFE marks the call sites where
// S may be a don't-care value of an idle lane (the window is at least 64 KB + 16 long: any 16-bit index stays inside).
template <int Q, bool SAFE = false>
__device__ __forceinline__ uint32_t tbl_gather(const Smem<Q> &sm, uint32_t S)
{
    const uint32_t idx = S >> 16;                 // no mask: see Cfg::SMEM_BYTES
    uint32_t rv;
    asm("ld.shared.u8 %0, [%1];" : "=r"(rv) : "r"(idx + sm.tbl_sa));
    return rv;
}

// tagged values: (value << VSHIFT) | don't-care bits of the index field
template <int Q> __device__ __forceinline__ uint32_t tag_value(int v) { return (uint32_t)v << Cfg<Q>::VSHIFT; }
template <int Q> __device__ __forceinline__ int untag(uint32_t x) { return (int)(x & 0xffffu); }
template <int Q> __device__ __forceinline__ uint32_t tag_max(uint32_t a, uint32_t b) { return __vmaxu2(a, b); }

// acc = max(acc, candidate of the word sum S): eq. (3)
template <int Q, bool SAFE = false>
__device__ __forceinline__ uint32_t lookup_max(const Smem<Q> &sm, uint32_t S, uint32_t acc)
{
    return __viaddmax_u16x2(S, tbl_gather<Q, SAFE>(sm, S), acc);
}

// Polls are relaxed loads (an acquire load also invalidates the L1 on every iteration); one acquire load
// orders the data reads after the flag has been seen.
__device__ __forceinline__ int ld_relaxed_gpu(const int *p)
{
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void wait_flag_ge(const int *flag, int v)
{
    if (ld_acquire_gpu(flag) >= v) return;
    unsigned ns = 64;
    while (ld_relaxed_gpu(flag) < v) { __nanosleep(ns); if (ns < 512) ns *= 2; }
    (void)ld_acquire_gpu(flag);
}

template <int Q>
__device__ __forceinline__ const uint8_t *rec_ptr(const Params &p, int sidx) { return p.recs + (size_t)sidx * Cfg<Q>::REC_BYTES; }

// bulk step (a4): acc[h][rr] = max over the 8 groups of block K, for columns cj + h*T/2 and rows rb*RPT+rr.
// acc is kept in the tagged form (value field + don't-care index bits); tag_max orders by value.
template <int Q>
__device__ __forceinline__ void product_accumulate(const Smem<Q> &sm, int buf, uint32_t (&acc)[2][Cfg<Q>::RPT], int cj, int rb)
{
    using C = Cfg<Q>;
    const uint32_t *PH = sm.stg + (size_t)buf * 2 * C::PANEL_WORDS;
    const uint32_t *PV = PH + C::PANEL_WORDS;
#pragma unroll 2
    for (int g = 0; g < 8; ++g) {
        const uint32_t X0 = PV[g * C::T + cj], X1 = PV[g * C::T + cj + C::HT];
        const uint32_t *wrow = PH + g * C::T + rb * C::RPT;
        uint32_t w[C::RPT];
        // the row words are warp-uniform: broadcast vector loads
        if constexpr (C::RPT % 4 == 0) {
#pragma unroll
            for (int r4 = 0; r4 < C::RPT / 4; ++r4) {
                const uint4 t4 = reinterpret_cast<const uint4 *>(wrow)[r4];
                w[4 * r4] = t4.x; w[4 * r4 + 1] = t4.y; w[4 * r4 + 2] = t4.z; w[4 * r4 + 3] = t4.w;
            }
        } else if constexpr (C::RPT % 2 == 0) {
#pragma unroll
            for (int r2 = 0; r2 < C::RPT / 2; ++r2) {
                const uint2 t2 = reinterpret_cast<const uint2 *>(wrow)[r2];
                w[2 * r2] = t2.x; w[2 * r2 + 1] = t2.y;
            }
        } else {
#pragma unroll
            for (int rr = 0; rr < C::RPT; ++rr) w[rr] = wrow[rr];
        }
#pragma unroll
        for (int rr = 0; rr < C::RPT; ++rr) {
            const uint32_t S0 = w[rr] + X0, S1 = w[rr] + X1;
            acc[0][rr] = lookup_max<Q>(sm, S0, acc[0][rr]);
            acc[1][rr] = lookup_max<Q>(sm, S1, acc[1][rr]);
        }
    }
}

// ---- mbarrier / bulk-copy primitives ----
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.release.cta.shared.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.acquire.cta.shared.b64 P1, [%0], %1, %2;\n"
        "@P1 bra.uni WAIT_DONE;\n"
        "bra.uni WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_addr(bar)), "r"(parity), "r"(20000u) : "memory");     // suspend-time hint (ns): park, do not spin
}

__device__ __forceinline__ void mbar_inval(uint64_t *bar)
{
    asm volatile("mbarrier.inval.shared.b64 [%0];" ::"r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
// Data that another CTA wrote with generic-proxy stores (st.global.cg + release flag) and that this thread is about
// to read through the async proxy (cp.async.bulk) needs a cross-proxy fence between the acquire of the flag and
// the copy (PTX memory model, "async proxy"); without it the two accesses are formally unordered.
__device__ __forceinline__ void fence_proxy_async_global()
{
    asm volatile("fence.proxy.async.global;" ::: "memory");
}
// TMA 1-D bulk copy global -> shared; completion is signalled on `bar` (complete_tx)
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gmem_src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_addr(smem_dst)), "l"(gmem_src), "r"(bytes), "r"(smem_addr(bar)) : "memory");
}

// ---- PROD task: merge the products of newly available middle blocks into the target's acc ----
template <int Q>
__device__ void run_prod(const Params &p, const Smem<Q> &sm, const SeqInfo &si, int I, int J, int s)
{
    using C = Cfg<Q>;
    const int tid = threadIdx.x;
    const int nt = si.nt;
    const int dp = J - I;
    const int S = nstages(dp, p.delta);
    const int hi = dp - 2 - s * p.delta;
    const int lo = max(hi - p.delta + 1, (dp + 1) / 2);
    const int sidx = si.sbase + tri_index(nt, I, J);
    const bool pact = tid < C::PTHR;             // threads beyond 4T only help with barriers (q < 8)
    const int cj = tid % C::HT, rb = pact ? tid / C::HT : 0;
    uint32_t acc[2][C::RPT];
#pragma unroll
    for (int rr = 0; rr < C::RPT; ++rr) acc[0][rr] = acc[1][rr] = 0;

    // K sequence: for m = lo..hi: K = I+m, then K = J-m (if different)
    const int nk_max = 2 * (hi - lo + 1);
    auto kth = [&](int e) -> int {           // e-th block of the sequence, or -1 for the duplicate
        const int m = lo + (e >> 1);
        const int K = (e & 1) ? (J - m) : (I + m);
        if ((e & 1) && (J - m == I + m)) return -1;
        return K;
    };
    // Warp-specialised operand pipeline: one producer warp (the first warp beyond the product threads) waits for
    // the operand tiles' flags and fetches PH(I,K), PV(K,J) with two TMA bulk copies per block into a NSTG-deep
    // ring; the product warps only ever wait on the ring's mbarriers, so flag and L2 latency stay off their path.
    constexpr int NPW = C::PTHR / 32;                      // product warps
    constexpr uint32_t PANEL_BYTES = C::PANEL_WORDS * 4;
    constexpr int NSTG = C::NSTG;
    uint64_t *full = sm.mbar + C::MB_PROD, *empty = full + 4;
    if (tid == 0) {
        for (int b = 0; b < NSTG; ++b) {
            mbar_inval(full + b); mbar_inval(empty + b);
            mbar_init(full + b, 1); mbar_init(empty + b, NPW);
        }
        mbar_inval(full + 3); mbar_init(full + 3, 1);          // the acc tile of the earlier stages has landed
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    const int warp = tid >> 5, lane = tid & 31;
    if (warp == NPW) {
        if (lane == 0) {
            int i = 0;
            for (int e = 0; e < nk_max; ++e) {
                const int K = kth(e);
                if (K < 0) continue;
                const int b = i % NSTG, k = i / NSTG;
                if (k >= 1) mbar_wait(empty + b, (uint32_t)(k - 1) & 1u);       // the product warps are done with the buffer
                const int s_ik = si.sbase + tri_index(nt, I, K), s_kj = si.sbase + tri_index(nt, K, J);
                wait_flag_ge(p.done + s_ik, 1);
                wait_flag_ge(p.done + s_kj, 1);
                fence_proxy_async_global();       // generic-proxy writes of other CTAs (acquired above) -> async-proxy reads below
                uint32_t *dst = sm.stg + (size_t)b * 2 * C::PANEL_WORDS;
                mbar_expect_tx(full + b, 2 * PANEL_BYTES);
                bulk_g2s(dst, rec_ptr<Q>(p, s_ik), PANEL_BYTES, full + b);                                   // PH of (I,K)
                bulk_g2s(dst + C::PANEL_WORDS, rec_ptr<Q>(p, s_kj) + PANEL_BYTES, PANEL_BYTES, full + b);     // PV of (K,J)
                ++i;
            }
            if (s != S - 1) {
                // earlier stages (they ran at earlier steps and own acc until their release): fetch their maxima
                wait_flag_ge(p.accstage + sidx, S - 1 - s);
                fence_proxy_async_global();
                mbar_expect_tx(full + 3, (uint32_t)(C::T * C::T * 2));
                bulk_g2s(sm.valraw, p.acc + (size_t)sidx * C::T * C::T, (uint32_t)(C::T * C::T * 2), full + 3);
            }
        }
    } else if (pact) {
        int i = 0;
        for (int e = 0; e < nk_max; ++e) {
            if (kth(e) < 0) continue;
            const int b = i % NSTG, k = i / NSTG;
            mbar_wait(full + b, (uint32_t)k & 1u);
            product_accumulate<Q>(sm, b, acc, cj, rb);
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + b);
            ++i;
        }
        if (s != S - 1) {
            mbar_wait(full + 3, 0u);
#pragma unroll
            for (int rr = 0; rr < C::RPT; ++rr) {
                const int16_t *row = sm.valraw + (rb * C::RPT + rr) * C::T + cj;
                acc[0][rr] = tag_max<Q>(acc[0][rr], tag_value<Q>((int)row[0]));
                acc[1][rr] = tag_max<Q>(acc[1][rr], tag_value<Q>((int)row[C::HT]));
            }
        }
    }
    int16_t *accg = p.acc + (size_t)sidx * C::T * C::T;
    if (pact) {
#pragma unroll
        for (int rr = 0; rr < C::RPT; ++rr) {
            int16_t *row = accg + (size_t)(rb * C::RPT + rr) * C::T + cj;
            __stcg(row, (int16_t)untag<Q>(acc[0][rr]));
            __stcg(row + C::HT, (int16_t)untag<Q>(acc[1][rr]));
        }
    }
    // the CTA barrier orders every thread's stores before thread 0's release (cumulative): no per-thread fence
    __syncthreads();
    if (tid == 0) st_release_gpu(p.accstage + sidx, S - s);
}

// ------------------------------------------------------------------------------------------------
// closure of one super-tile (steps a3, a5, a6, a7 inside the CTA)
//
// Local coordinates: rows a = 0..T-1 (a = T-1 is the bottom row), columns c = 0..T-1; the super-tile
// is 8 x 8 q-tiles (A,B) of Q x Q cells.  q-tile (A,B) needs (A+1,B) and (A,B-1): the q-tiles of one
// anti-diagonal u = (7-A)+B are independent and run together as a "macro-step" (15 per super-tile;
// PAPER.md:223-245 wavefront, PAPER.md:291 tiles of one diagonal are independent).  The CTA's warps take
// roles: closure warps (G q-tiles side by side per warp, Q lanes each), mini helpers,
// loaders, late-product helpers, publishers; the closure warps and the mini helpers meet at a named
// barrier twice per macro-step, everything else is ordered by shared-memory mbarriers.
//
// Per q-tile:
//  (M) every group that is complete for the whole q-tile -- z in [A+1, 7] of block I (column words of the
//      q-tiles below, row words of (I,I)) and z in [8, 8+B-1] of block J (row words of the q-tiles to the
//      left, column words of (J,J)) -- is one lookup per cell (full groups).  The two
//      groups that were finished in the previous macro-step are looked up in phase F (qtile_fresh_merge),
//      the older ones one macro-step ahead by the mini helpers (into val3).
//  (C) cell wavefront, lane y <-> column BQ+y, 2Q skewed steps, lane y one row below lane y-1.  Of all
//      candidates of cell (a,c) only two depend on the previous step:
//        left  = v(a,c-1)  (tail split t = c-1: M(r,c-1) + M(c-1,c), M(c-1,c) = 0)   -- one shuffle
//        below = v(a+1,c)  (head split t = r+1: M(r,r+1) + M(r+1,c), M(r,r+1) = 0)   -- own register.
//      Everything else of the NEXT cell (a-1,c) -- val (bulk + mini-products), b + D(i+1,j-1)
//      (PAPER.md:135), the head lookup (running column word Xp over rows >= a+1 of the q-tile with the
//      row word of group A of block I) and the tail lookup (row word of row a-1 through column c-2,
//      from lane y-2, with the column word of group B of block J) -- is computed during the step
//      ("oldx") and enters v(a-1,c) one step later: the dependent chain of a step is shuffle -> max.
//      Head and tail are the paper's residual loops done as masked
//      lookups: not yet known difference bits are zero (DESIGN.md 4.3 proves this is exact).
// DIAG (I == J): row and column words are both the tile's own (z < 8 only); macro-steps start at u = 7;
// in q-tile (B,B) head and tail are ONE lookup (row word through c-2, Xp); cells with c-a <= 1 are 0.
// ------------------------------------------------------------------------------------------------

// Complete-group lookups for the Q x Q cells of q-tile (A,B), all 32 lanes: for z in [zlo, zhi],
// val[a][c] = max(val[a][c], lookup(W[z*wp + a] + X[z*xp + c])).  Used for the mini-products of the
// closure (W = Wst, X = Xst) and for the late products (operand panels of the neighbouring blocks).
template <int Q>
__device__ __forceinline__ void qtile_groups(const Smem<Q> &sm, int A, int B, const uint32_t *W, int wp, const uint32_t *X, int xp,
                                             int zlo, int zhi, int lane, bool merge2 = false, bool out3 = false)
{
    using C = Cfg<Q>;
    constexpr int VP = C::VP;
    constexpr int RS = (32 / Q > Q) ? Q : 32 / Q;        // row slots
    constexpr int NX = (Q + RS - 1) / RS;                // rows per lane
    const int my = lane % Q, xr = lane / Q;
    if ((zlo > zhi && !merge2) || xr >= RS) return;
    const int mc = B * Q + my;
    const int abot = A * Q + Q - 1;
    uint32_t best[NX];
#pragma unroll
    for (int i = 0; i < NX; ++i) best[i] = 0;
#pragma unroll 2
    for (int z = zlo; z <= zhi; ++z) {
        const uint32_t Xw = X[z * xp + mc];
#pragma unroll
        for (int i = 0; i < NX; ++i) {
            const int x = xr + i * RS;
            const int a = abot - (x < Q ? x : 0);
            best[i] = lookup_max<Q>(sm, W[z * wp + a] + Xw, best[i]);
        }
    }
#pragma unroll
    for (int i = 0; i < NX; ++i) {
        const int x = xr + i * RS;
        if (x < Q && out3) {
            sm.val3[(abot - x) * C::VP2 + mc] = (int16_t)untag<Q>(best[i]);      // written once per cell
        } else if (x < Q) {
            int16_t *cell = sm.val + (abot - x) * VP + mc + 1;
            int v = max((int)*cell, untag<Q>(best[i]));
            if (merge2) v = max(v, (int)sm.val2[(abot - x) * C::VP2 + mc]);      // late products of block I+1
            *cell = (int16_t)v;
        }
    }
}

// (C) phase of q-tile (A,B): 2Q unrolled skewed steps; every address is lane base + immediate.
// MERGED: q-tile (B,B) of a diagonal super-tile (head and tail are one lookup; c-a = s-Q+1 for every lane).
template <int Q, bool DIAG, bool MERGED>
__device__ __forceinline__ void qtile_wave(const Smem<Q> &sm, int A, int B, int lane, bool own)
{
    using C = Cfg<Q>;
    constexpr int TP = C::TP, VP = C::VP;
    constexpr uint32_t FULL = 0xffffffffu;
    constexpr int ZOFF = DIAG ? 0 : 8;
    const int y = lane % Q;                              // lane group lane/Q runs q-tile (A,B); !own: shadow, stores nothing
    const bool firstcol = (y == 0), lastcol = (y == Q - 1);
    const int src1 = firstcol ? lane : lane - 1, src2 = (y >= 2) ? lane - 2 : lane;
    const uint32_t w2mask = (y >= 2) ? FULL : 0u;
    const int c = B * Q + y;
    const int abot = A * Q + Q - 1;
    uint32_t khy = ((uint32_t)C::TBL_PITCH << (y > 0 ? y - 1 : 0)) << C::ISHIFT;   // index weight of my horizontal difference bit
    if constexpr (C::TERN) {                             // 3^(y-1) instead of 2^(y-1)
        khy = 1u << C::ISHIFT;
#pragma unroll
        for (int k = 1; k < Q - 1; ++k) if (k < y) khy *= 3u;
    }
    uint32_t w3 = 0;                                     // TERN: index weight 3^(Q-1-x) of the next vertical difference bit
    const int sh0 = C::ISHIFT + Q - 2 + y;                  // vertical bit of row x = s-y sits at sh0 - (s-1) (sh0 <= 31)
    const uint32_t XJ = MERGED ? 0u : sm.Xst[(ZOFF + B) * TP + c];
    uint32_t pms = 0;                                    // bit (x + y) <-> row x pairs with my column
    {
        const int want = 3 - (int)sm.codeC[c];
#pragma unroll
        for (int x = 0; x < Q; ++x) pms |= (uint32_t)((int)sm.codeR[abot - x] == want) << x;
        pms <<= y;
    }
    int16_t *vb = sm.val + (abot + y) * VP + c + 1;                 // vb[-s*VP]  = val[a][c],  a = abot + y - s
    const uint32_t *wb = sm.Wst + A * TP + abot + y - 1;            // wb[-s]     = Wst[A][a-1]
    uint32_t *wo = sm.Wst + (ZOFF + B) * TP + abot + y;             // wo[-s]     = own row word of row a
    int vprev = 0;
    uint32_t wout = 0, xbits = 0, vsh = 0;
    // Operands that do not depend on this wavefront (the head row word, the prepared value of the next cell, the
    // left neighbour's column for lane 0, the cell below the q-tile) are loaded one step ahead: a single warp
    // issues in order, so a load placed next to its use would add its 29 cycles to every step.
    const int vbelow = sm.val[(abot + 1) * VP + c + 1];
    uint32_t w_nxt = wb[1];
    int o_nxt = vb[0], lv_nxt = vb[VP - 1];
    // The two lookups of a step are only consumed one step later (they belong to the NEXT cell), so they are
    // carried as pending (word sum, table byte) pairs and folded in after the next step's shuffles have been
    // issued: gather latency and shuffle latency overlap instead of adding up.
    uint32_t hS = 0, hR = 0, tS = 0, tR = 0;
    int o_pend = 0;
#pragma unroll
    for (int s = -1; s <= 2 * Q - 2; ++s) {
        const int x_lo = s - (Q - 1);                               // rows touched this step: x in [x_lo, s]
        const uint32_t w_cur = w_nxt;
        const int o_cur = o_nxt, lv_cur = lv_nxt;
        if (s < 2 * Q - 2) { w_nxt = wb[-(s + 1)]; o_nxt = vb[-(s + 2) * VP]; lv_nxt = vb[-(s + 1) * VP - 1]; }
        const uint32_t phS = hS, phR = hR, ptS = tS, ptR = tR;      // the lookups issued in the previous step (my cell's)
        // ---- head lookup of the NEXT cell: running column word (rows >= a+1) x row word of group A of block I
        uint32_t Xp = xbits + vsh;
        if (s + 1 < Q && y > s) Xp = 0;                             // not in the q-tile yet: no row of it lies below
        if (!MERGED) { hS = w_cur + Xp; hR = tbl_gather<Q, true>(sm, hS); }
        // ---- receive from the left
        int Lv = __shfl_sync(FULL, vprev, src1);                    // v(a, c-1)
        const uint32_t Lw = __shfl_sync(FULL, wout, src1);          // row a   through column c-1
        const uint32_t Lw2 = __shfl_sync(FULL, wout, src2) & w2mask;   // row a-1 through column c-2
        if (firstcol) Lv = lv_cur;                                  // column c-1 belongs to the q-tile on the left
        // ---- the cell (a3 init + a5 fresh splits)
        // The pending lookups are folded in with the direct candidates as their accumulator: their consumers then
        // depend on the shuffle result and cannot be scheduled -- with their wait for the gathers -- before the
        // shuffles are issued (a single warp issues in order).
        uint32_t best = tag_value<Q>(max(max(o_pend, vprev), Lv));
        if (!MERGED) best = __viaddmax_u16x2(phS, phR, best);
        best = __viaddmax_u16x2(ptS, ptR, best);
        int v = untag<Q>(best);
        if (s + 1 < Q && y == s + 1) v = vbelow;                    // pre-step (x = -1): the cell below the q-tile
        if (MERGED && s - (Q - 1) <= 1) v = 0;                      // D(i,i) = D(i,i-1) = 0
        const bool live = own && (unsigned)(s - y) < (unsigned)Q;
        RNA4R_CHECK(!live || ((unsigned)(v - Lv) <= 1u && (s - y == 0 || (unsigned)(v - vprev) <= 1u)));   // Lemma 1 against the left and the lower cell
        if (live) vb[-s * VP] = (int16_t)v;
        // ---- tail lookup of the NEXT cell: row word of row a-1 through column c-2 x column word of group B of block J
        tS = Lw2 + (MERGED ? Xp : XJ);
        tR = tbl_gather<Q, true>(sm, tS);
        // ---- step a6, horizontal: my row word = neighbour's word | my difference bit
        const uint32_t vnew = tag_value<Q>(v);
        const uint32_t wme = firstcol ? vnew : (Lw + (uint32_t)(v - Lv) * khy);
        if (live && lastcol) {
            wo[-s] = wme;
            if (DIAG) wo[-s + 8 * TP] = wme;
        }
        // ---- the rest of the next cell's candidates: prepared value, b(S_i,S_j) + D(i+1,j-1)
        o_pend = max(o_cur, Lv + (int)((pms >> ((s + 1) & 31)) & 1u));
        // ---- step a6, vertical: the column word now starts at row a (anchor v, bit of the pair (a, a+1))
        {
            if constexpr (C::TERN) {
                // a column word without set bits has the index part sum_k 3^k (digit 1 = "no difference"); the bit of
                // the pair (row x, row x-1) takes 3^(Q-1-x) away.  The weight goes down by a factor 3 per row (an exact
                // division; beyond the top row of the q-tile it runs out, those lanes are not live).
                if (y <= s - 1) { xbits -= (uint32_t)(v - vprev) * w3; w3 = __umulhi(w3, 0xAAAAAAABu) >> 1; }
                else { xbits = C::TERN_C0 << C::ISHIFT; w3 = C::pow3(Q - 2) << C::ISHIFT; }
            } else {
                const uint32_t dbit = ((uint32_t)(v - vprev) << sh0) >> ((s >= 1 ? s - 1 : 0) & 31);   // used for x >= 1 only
                xbits = (y <= s - 1) ? ((xbits | dbit) & C::VMASK) : 0u;     // x >= 1
            }
            vsh = vnew;
        }
        if (x_lo >= 0 && live && y == x_lo) sm.Xst[A * TP + c] = xbits + vsh;    // x = Q-1: the column word is complete
        vprev = v; wout = wme;
    }
}

// Operand panels of the late products, in the staging area (pitch T): rows of the left tile (I,J-1),
// column panel of (J-1,J), row panel of (I,I+1), columns of the tile below (I+1,J).
template <int Q> __device__ __forceinline__ uint32_t *panel_ZW(const Smem<Q> &sm) { return sm.stg; }
template <int Q> __device__ __forceinline__ uint32_t *panel_XJ1(const Smem<Q> &sm) { return sm.stg + Cfg<Q>::PANEL_WORDS; }
template <int Q> __device__ __forceinline__ uint32_t *panel_WI1(const Smem<Q> &sm) { return sm.stg + 2 * Cfg<Q>::PANEL_WORDS; }
template <int Q> __device__ __forceinline__ uint32_t *panel_YX(const Smem<Q> &sm) { return sm.stg + 3 * Cfg<Q>::PANEL_WORDS; }

struct CloseCtx {
    int dp;              // J - I
    uint32_t parity;     // phase of this closure's mbarriers
    const uint8_t *recZ; // record of the left tile (I,J-1)
    const uint8_t *recY; // record of the tile below (I+1,J)
    const uint8_t *recC; // record of the corner tile (I+1,J-1), or NULL (dp < 2: below the diagonal, value 0)
    uint8_t *recX;       // record of this tile
    const int *rowprogZ, *colprogY, *doneC;
    int *rowprogX, *colprogX;
    unsigned long long *prof; // trace record of this closure, or NULL
    unsigned long long *ev;   // fine trace of this closure (RNA4R_TRACE_WORDS > 8), else NULL
};
#define RNA4R_EV(cc, idx) do { if (RNA4R_TRACE_WORDS > 8 && (cc).ev && lane == 0) (cc).ev[idx] = global_timer_ns(); } while (0)

// waits until *flag >= v; returns the value seen (clamped to 8: the flags count q-rows / q-columns)
__device__ __forceinline__ int warp_wait_flag_ge(const int *flag, int v, int lane)
{
    int have = 0;
    if (lane == 0) {
        while ((have = ld_acquire_gpu(flag)) < v) __nanosleep(32);     // every poll is an acquire: no second round trip once the flag is seen
    }
    __syncwarp();                                                      // orders the other lanes' data loads after lane 0's acquire
    have = __shfl_sync(0xffffffffu, have, 0);
    return have < 8 ? have : 8;
}

__device__ __forceinline__ void named_bar_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// q-tile t of macro-step u (anti-diagonal (7-A)+B = u), counted from the bottom-left
__device__ __forceinline__ void qtile_of(int u, int t, int &A, int &B)
{
    const int Amax = min(7, 14 - u);
    A = Amax - t;
    B = u - (7 - A);
}
__device__ __forceinline__ int qtile_count(int u) { return min(7, 14 - u) - max(0, 7 - u) + 1; }

// Before the cell wavefronts of a macro-step, everything that is known about its q-tiles is folded into val[][]:
// the late products of block I+1 (val2), the older complete groups prepared by the mini helpers (val3) and the
// two complete groups that were only finished in the previous macro-step -- the lowest and the highest z of the
// q-tile's range [A+1, ZOFF+B-1] (column word of the q-tile below, row word of the q-tile to the left).
// One warp per q-tile, all 32 lanes (the closure warps and the mini helpers share the q-tiles of the macro-step).
template <int Q, bool DIAG>
__device__ __forceinline__ void qtile_fresh_merge(const Smem<Q> &sm, int A, int B, int lane, bool use2)
{
    using C = Cfg<Q>;
    constexpr int TP = C::TP, VP = C::VP, VP2 = C::VP2;
    constexpr int ZOFF = DIAG ? 0 : 8;
    constexpr int RS = (32 / Q > Q) ? Q : 32 / Q;        // row slots
    constexpr int NX = (Q + RS - 1) / RS;                // rows per lane
    const int my = lane % Q, xr = lane / Q;
    if (xr >= RS) return;
    const int c = B * Q + my;
    const int abot = A * Q + Q - 1;
    const int lo = A + 1, hi = ZOFF + B - 1;
    const bool has1 = lo <= hi, has2 = hi > lo;
    const uint32_t X1 = has1 ? sm.Xst[lo * TP + c] : 0u;
    const uint32_t X2 = has2 ? sm.Xst[hi * TP + c] : 0u;
    const uint32_t *w1 = sm.Wst + (has1 ? lo : 0) * TP;
    const uint32_t *w2 = sm.Wst + (has2 ? hi : 0) * TP;
    const uint32_t m1 = has1 ? 0xffffffffu : 0u, m2 = has2 ? 0xffffffffu : 0u;
#pragma unroll
    for (int i = 0; i < NX; ++i) {
        const int x = xr + i * RS;
        if (x < Q) {
            const int a = abot - x;
            int v = max((int)sm.val[a * VP + c + 1], (int)sm.val3[a * VP2 + c]);
            if (use2) v = max(v, (int)sm.val2[a * VP2 + c]);
            const uint32_t b1 = lookup_max<Q>(sm, (w1[a] & m1) + X1, 0u);     // a zero pair looks up R[0][0] = 0
            const uint32_t b2 = lookup_max<Q>(sm, (w2[a] & m2) + X2, b1);
            v = max(v, untag<Q>(b2));
            sm.val[a * VP + c + 1] = (int16_t)v;
        }
    }
}

// what macro-step u of an off-diagonal super-tile newly touches: q-row 7-u enters at column 0 (left half of
// its late products, left edge), q-column u enters at row 7 (lower half, bottom edge); four macro-steps later
// they reach the other half
template <int Q>
__device__ __forceinline__ void step_waits(const Smem<Q> &sm, const CloseCtx &cc, int u)
{
    using C = Cfg<Q>;
    if (u <= 11) mbar_wait(sm.mbar + C::MB_STEPIN + u, cc.parity);
}

// phase F of macro-step u, step warp sw of NWV+NMH
template <int Q, bool DIAG>
__device__ __forceinline__ void macro_fresh(const Smem<Q> &sm, const CloseCtx &cc, int u, int sw, int lane)
{
    using C = Cfg<Q>;
    const int cnt = qtile_count(u);
    for (int t = sw; t < cnt; t += C::NWV + C::NMH) {
        int A, B;
        qtile_of(u, t, A, B);
        qtile_fresh_merge<Q, DIAG>(sm, A, B, lane, !DIAG && cc.dp >= 3);
    }
}

// closure warp w of NWV: G q-tiles of the current anti-diagonal side by side, macro-step by macro-step.
// A macro-step is phase F (fresh merge, all step warps) | barrier | phase W (cell wavefronts here, older groups
// of the next macro-step in the mini helpers) | barrier.
template <int Q, bool DIAG>
__device__ __forceinline__ void close_wave(const Smem<Q> &sm, const CloseCtx &cc, int w, int lane)
{
    using C = Cfg<Q>;
    const int j = lane / Q;
    long long pf_merge = 0, pf_wave = 0, pf_bar = 0;
    named_bar_sync(1, C::STEP_THREADS);                 // val3 is cleared
#pragma unroll 1
    for (int u = DIAG ? 7 : 0; u < 15; ++u) {
        const long long c0 = clock64();
        macro_fresh<Q, DIAG>(sm, cc, u, w, lane);
        named_bar_sync(1, C::STEP_THREADS);
        const long long c1 = clock64();
        const int cnt = qtile_count(u);
        const int t = w * C::G + j;
        const bool own = (j < C::G) && (t < cnt);
        int A, B;
        qtile_of(u, own ? t : 0, A, B);
        if (w * C::G < cnt) {
            if (DIAG && u == 7) qtile_wave<Q, true, true>(sm, A, B, lane, own);
            else qtile_wave<Q, DIAG, false>(sm, A, B, lane, own);
        }
        const long long c2 = clock64();
        named_bar_sync(1, C::STEP_THREADS);
        const long long c3 = clock64();
        pf_merge += c1 - c0; pf_wave += c2 - c1; pf_bar += c3 - c2;
        if (w == 0 && lane == 0) mbar_arrive(sm.mbar + C::MB_STEP + u);
        if (w == 0) RNA4R_EV(cc, 8 + u);
    }
    if (cc.prof && w == 0 && lane == 0)
        cc.prof[7] = ((unsigned long long)(pf_merge & 0x1fffff)) | ((unsigned long long)(pf_wave & 0x1fffff) << 21) | ((unsigned long long)(pf_bar & 0x1fffff) << 42);
}

// mini helper h of NMH: shares phase F; in phase W, while the closure warps run the cell wavefronts of
// macro-step u, the older complete groups z in [A+2, ZOFF+B-2] of the q-tiles of macro-step u+1 (all finished
// by macro-step u-1) -> val3
template <int Q, bool DIAG>
__device__ __forceinline__ void close_mini_helper(const Smem<Q> &sm, const CloseCtx &cc, int h, int lane)
{
    using C = Cfg<Q>;
    constexpr int ZOFF = DIAG ? 0 : 8;
    {
        uint32_t *z = reinterpret_cast<uint32_t *>(sm.val3);
        for (int e = h * 32 + lane; e < C::VAL2_BYTES / 4; e += C::NMH * 32) z[e] = 0;
    }
    // What a macro-step needs from the loaders and late-product helpers is awaited by mini helper 0 alone, one
    // macro-step ahead and after its own work (an mbarrier test costs ~90 cycles even when it has completed);
    // the named barrier that closes the macro-step hands the guarantee to everybody.
    if (!DIAG && h == 0) step_waits<Q>(sm, cc, 0);
    named_bar_sync(1, C::STEP_THREADS);
#pragma unroll 1
    for (int u = DIAG ? 7 : 0; u < 15; ++u) {
        macro_fresh<Q, DIAG>(sm, cc, u, C::NWV + h, lane);
        named_bar_sync(1, C::STEP_THREADS);
        if (u + 1 < 15) {
            const int cnt = qtile_count(u + 1);
            for (int t = h; t < cnt; t += C::NMH) {
                int A, B;
                qtile_of(u + 1, t, A, B);
                qtile_groups<Q>(sm, A, B, sm.Wst, C::TP, sm.Xst, C::TP, A + 2, ZOFF + B - 2, lane, false, true);
            }
            if (!DIAG && h == 0) step_waits<Q>(sm, cc, u + 1);
        }
        named_bar_sync(1, C::STEP_THREADS);
    }
}

// Loader loop shared by the row and the column loader.  `unit` counts q-rows from the bottom (q-columns from the
// left) in publishing order; unit k covers words [g][first(k) .. first(k)+Q) of the neighbour's panel `src` (pitch
// T) and Q edge values.  Up to two published units are fetched per iteration, and the next flag read is issued
// while their data is still in flight, so an iteration costs one L2 round trip instead of two.
template <int Q, typename FirstOf, typename EdgeDst>
__device__ __forceinline__ void loader_loop(const int *flag, const uint32_t *src, const uint16_t *esrc, uint32_t *dst, FirstOf first_of,
                                            EdgeDst edge_dst, uint64_t *bars, const CloseCtx &cc, int ev0, int lane)
{
    using C = Cfg<Q>;
    constexpr int T = C::T;
    constexpr int NW = (8 * Q + 31) / 32;
    int have = warp_wait_flag_ge(flag, 1, lane);
    int loaded = 0;
    while (loaded < 8) {
        const int hi = min(have, loaded + 2);
        uint32_t w[2][NW];
        uint16_t ev[2];
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            const int k0 = first_of(min(loaded + r, 7));
#pragma unroll
            for (int i = 0; i < NW; ++i) {
                const int e = lane + 32 * i;
                w[r][i] = (e < 8 * Q && loaded + r < hi) ? __ldcg(src + (e / Q) * T + k0 + e % Q) : 0u;
            }
            ev[r] = (lane < Q && loaded + r < hi) ? __ldcg(esrc + k0 + lane) : (uint16_t)0;
        }
        int next = 8;
        if (hi < 8 && lane == 0) next = ld_acquire_gpu(flag);         // in flight together with the data
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            if (loaded + r < hi) {
                const int k0 = first_of(loaded + r);
#pragma unroll
                for (int i = 0; i < NW; ++i) {
                    const int e = lane + 32 * i;
                    if (e < 8 * Q) dst[(e / Q) * T + k0 + e % Q] = w[r][i];
                }
                if (lane < Q) *edge_dst(k0 + lane) = (int16_t)ev[r];
            }
        }
        __syncwarp();
        for (int k = loaded; k < hi; ++k) {
            if (lane == 0) mbar_arrive(bars + first_of(k) / Q);
            RNA4R_EV(cc, ev0 + first_of(k) / Q);
        }
        loaded = hi;
        if (loaded < 8) {
            __syncwarp();                                              // lane 0's acquire of `next` precedes everybody's next data loads
            have = min(__shfl_sync(0xffffffffu, next, 0), 8);
            if (have <= loaded) have = warp_wait_flag_ge(flag, loaded + 1, lane);
        }
    }
}

// helper warp: columns of the tile below, q-column by q-column as it publishes them (column words for the
// late products, top-row values = my bottom edge), and the corner value
template <int Q>
__device__ __forceinline__ void close_col_loader(const Smem<Q> &sm, const CloseCtx &cc, int lane)
{
    using C = Cfg<Q>;
    constexpr int T = C::T, VP = C::VP;
    const uint32_t *pv = reinterpret_cast<const uint32_t *>(cc.recY) + C::PANEL_WORDS;
    const uint16_t *etop = reinterpret_cast<const uint16_t *>(cc.recY + 2 * C::PANEL_WORDS * 4);
    uint32_t *YX = panel_YX<Q>(sm);
    if (lane == 0) {
        // corner M((I+1)T, JT-1) = top row of (I+1,J-1) at its last column
        int corner = 0;
        if (cc.recC) {
            wait_flag_ge(cc.doneC, 1);
            corner = __ldcg(reinterpret_cast<const uint16_t *>(cc.recC + 2 * C::PANEL_WORDS * 4) + T - 1);
        }
        sm.val[T * VP] = (int16_t)corner;
    }
    loader_loop<Q>(cc.colprogY, pv, etop, YX, [](int k) { return k * Q; },
                   [&](int c) { return sm.val + T * VP + c + 1; }, sm.mbar + C::MB_COL, cc, 144, lane);
}

// helper warp: rows of the left tile, q-row by q-row as it publishes them (row words for the late
// products, right-column values = my left edge)
template <int Q>
__device__ __forceinline__ void close_row_loader(const Smem<Q> &sm, const CloseCtx &cc, int lane)
{
    using C = Cfg<Q>;
    constexpr int T = C::T, VP = C::VP;
    const uint32_t *ph = reinterpret_cast<const uint32_t *>(cc.recZ);
    const uint16_t *eright = reinterpret_cast<const uint16_t *>(cc.recZ + 2 * C::PANEL_WORDS * 4) + T;
    uint32_t *ZW = panel_ZW<Q>(sm);
    loader_loop<Q>(cc.rowprogZ, ph, eright, ZW, [](int k) { return (7 - k) * Q; },
                   [&](int a) { return sm.val + a * VP; }, sm.mbar + C::MB_ROW, cc, 136, lane);
}

// helper warps: publish the tile q-column by q-column (which = 0) and q-row by q-row (which = 1) (step a6
// output): column words and top-row values of q-column B once q-tile (0,B) is done, row words and right-column
// values of q-row A once q-tile (A,7) is done -- both are on anti-diagonal 7+i.
template <int Q>
__device__ __forceinline__ void close_publisher(const Smem<Q> &sm, const CloseCtx &cc, int which, int lane)
{
    using C = Cfg<Q>;
    constexpr int T = C::T, TP = C::TP, VP = C::VP;
    uint32_t *ph = reinterpret_cast<uint32_t *>(cc.recX);
    uint32_t *pv = ph + C::PANEL_WORDS;
    uint16_t *edge = reinterpret_cast<uint16_t *>(cc.recX + 2 * C::PANEL_WORDS * 4);
    for (int i = 0; i < 8; ++i) {
        mbar_wait(sm.mbar + C::MB_STEP + 7 + i, cc.parity);
        if (which == 0) {
            const int B = i;
            for (int e = lane; e < 8 * Q; e += 32) {
                const int g = e / Q, k = B * Q + e % Q;
                __stcg(pv + g * T + k, sm.Xst[g * TP + k]);
            }
            if (lane < Q) __stcg(edge + B * Q + lane, (uint16_t)sm.val[B * Q + lane + 1]);           // top row  M(I*T, c)
            __syncwarp();
            if (lane == 0) st_release_gpu(cc.colprogX, B + 1);
            RNA4R_EV(cc, 224 + B);
        } else {
            const int A = 7 - i;
            for (int e = lane; e < 8 * Q; e += 32) {
                const int g = e / Q, k = A * Q + e % Q;
                __stcg(ph + g * T + k, sm.Wst[(8 + g) * TP + k]);
            }
            if (lane < Q) __stcg(edge + T + A * Q + lane, (uint16_t)sm.val[(A * Q + lane) * VP + T]);   // right column M(r, J*T+T-1)
            __syncwarp();
            if (lane == 0) st_release_gpu(cc.rowprogX, 8 - A);
            RNA4R_EV(cc, 216 + A);
        }
    }
}

// Late products: the two middle blocks K = J-1 and K = I+1 whose panels are only being finished now.
// One max-plus product of Q rows x T columns (row_late: rows of q-row A of the left tile x column panel of
// (J-1,J)) or T rows x Q columns (col_late: row panel of (I,I+1) x columns of q-column B of the tile below)
// over the 8 groups of the block; a lane owns one column (row) and NR rows (columns), so the words of the
// short side are warp-uniform broadcast loads, as in the bulk product.
template <int Q>
__device__ __forceinline__ void late_strip(const Smem<Q> &sm, const uint32_t *U, int u0, const uint32_t *L, int l0, int l1, int16_t *out,
                                           int out_us, int out_ls, bool domax, int lane)
{
    // U[g*T + u0 + i], i < Q: the uniform side; L[g*T + l], l0 <= l < l1: the lane side; out[(u0+i)*out_us + l*out_ls]
    using C = Cfg<Q>;
    constexpr int T = C::T;
    for (int l = l0 + lane; l < l1; l += 32) {
        uint32_t acc[Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) acc[i] = 0;
#pragma unroll 2
        for (int g = 0; g < 8; ++g) {
            const uint32_t Lw = L[g * T + l];
            const uint32_t *u = U + g * T + u0;
#pragma unroll
            for (int i = 0; i < Q; ++i) acc[i] = lookup_max<Q>(sm, u[i] + Lw, acc[i]);
        }
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            int16_t *cell = out + (u0 + i) * out_us + l * out_ls;
            const int v = untag<Q>(acc[i]);
            *cell = (int16_t)(domax ? max((int)*cell, v) : v);
        }
    }
}

// helper warps: q-row A as soon as the loader has it (rows of the left tile): block K = J-1, into val;
// warp h takes the columns of q-columns 4h..4h+3
template <int Q>
__device__ __forceinline__ void close_row_late(const Smem<Q> &sm, const CloseCtx &cc, int h, int lane)
{
    using C = Cfg<Q>;
    if (cc.dp == 2)       // K = J-1 = I+1: both operands arrive now; wait for my columns of the tile below
        for (int B = 4 * h; B < 4 * h + 4; ++B) mbar_wait(sm.mbar + C::MB_COL + B, cc.parity);
    for (int A = 7; A >= 0; --A) {
        mbar_wait(sm.mbar + C::MB_ROW + A, cc.parity);
        if (cc.dp >= 2)
            late_strip<Q>(sm, panel_ZW<Q>(sm), A * Q, cc.dp == 2 ? panel_YX<Q>(sm) : panel_XJ1<Q>(sm), 4 * Q * h, 4 * Q * h + 4 * Q,
                          sm.val + 1, C::VP, 1, true, lane);
        __syncwarp();
        if (lane == 0) mbar_arrive(sm.mbar + C::MB_STEPIN + (h == 0 ? 7 - A : 11 - A));
        if (h == 0) RNA4R_EV(cc, 152 + A);
    }
}

// helper warps: q-column B as soon as the loader has it (columns of the tile below): block K = I+1, into val2;
// warp h takes the rows of q-rows 4h..4h+3 (h = 1, the lower half, is needed first)
template <int Q>
__device__ __forceinline__ void close_col_late(const Smem<Q> &sm, const CloseCtx &cc, int h, int lane)
{
    using C = Cfg<Q>;
    for (int B = 0; B < 8; ++B) {
        mbar_wait(sm.mbar + C::MB_COL + B, cc.parity);
        if (cc.dp >= 3)
            late_strip<Q>(sm, panel_YX<Q>(sm), B * Q, panel_WI1<Q>(sm), 4 * Q * h, 4 * Q * h + 4 * Q, sm.val2, 1, C::VP2, false, lane);
        __syncwarp();
        if (lane == 0) mbar_arrive(sm.mbar + C::MB_STEPIN + (h == 1 ? B : B + 4));
        if (h == 1) RNA4R_EV(cc, 160 + B);
    }
}

// ---- CLOSE task ----
template <int Q>
__device__ void run_close(const Params &p, const Smem<Q> &sm, const SeqInfo &si, int seq, int I, int J)
{
    using C = Cfg<Q>;
    constexpr int T = C::T;
    const int tid = threadIdx.x;
    const int nt = si.nt;
    const int dp = J - I;
    const int sidx = si.sbase + tri_index(nt, I, J);
    unsigned long long *tr = (p.trace && sidx < p.trace_tiles) ? p.trace + (size_t)sidx * RNA4R_TRACE_WORDS : nullptr;
    if (tr && tid == 0) { tr[0] = global_timer_ns(); tr[6] = ((unsigned long long)I << 32) | (unsigned)J; }

    // codes of the rows r = I*T + a (base S[r]) and of the columns c = J*T + jj (base S[c-1])
    if (tid < T) {
        sm.codeR[tid] = p.codes[si.cbase + I * T + tid];
        const int c = J * T + tid;
        sm.codeC[tid] = (c >= 1) ? p.codes[si.cbase + c - 1] : (int8_t)4;
    }
    // roles by warp, counted from the top: the SM's issue arbiter favours high warp ids, and the closure
    // warps carry the critical path
    // co-resident CTAs (block index apart by a multiple of the SM count) rotate the roles by two warps, so that
    // their closure warps land on different SM sub-partitions (warp id mod 4)
    constexpr int NWARP = C::NTHR / 32;
    const int rot = 2 * ((blockIdx.x / p.sm_count) % 2);
    const int warp = ((NWARP - 1) - (tid >> 5) + NWARP - rot) % NWARP, lane = tid & 31;
    CloseCtx cc;
    cc.dp = dp;
    cc.parity = (uint32_t)sm.misc[1] & 1u;    // closures this CTA has run so far: phase of its mbarriers
    cc.recX = const_cast<uint8_t *>(rec_ptr<Q>(p, sidx));
    cc.rowprogX = p.rowprog + sidx; cc.colprogX = p.colprog + sidx;
    cc.prof = tr;
    cc.ev = (RNA4R_TRACE_WORDS > 8) ? tr : nullptr;
    cc.recZ = cc.recY = cc.recC = nullptr; cc.rowprogZ = cc.colprogY = cc.doneC = nullptr;

    if (dp == 0) {
        // diagonal super-tile: everything starts from zero; no neighbour, no late product
        for (int e = tid; e < C::VAL_BYTES / 4; e += C::NTHR) reinterpret_cast<uint32_t *>(sm.valraw)[e] = 0;
        for (int e = tid; e < C::WROWS * C::TP; e += C::NTHR) { sm.Wst[e] = 0; sm.Xst[e] = 0; }
        __syncthreads();
        if (warp < C::NWV) close_wave<Q, true>(sm, cc, warp, lane);
        else if (warp < C::NWV + C::NMH) close_mini_helper<Q, true>(sm, cc, warp - C::NWV, lane);
        else if (warp == C::NWV + C::NMH) {
            // keep the phases of the barriers a diagonal super-tile does not use in step
            if (lane < 16) mbar_arrive(sm.mbar + C::MB_ROW + lane);
            if (lane < 12) for (int k = 0; k < C::stepin_count(lane); ++k) mbar_arrive(sm.mbar + C::MB_STEPIN + lane);
            if (lane < 7) mbar_arrive(sm.mbar + C::MB_STEP + lane);
        }
        __syncthreads();
        if (tr && tid == 0) tr[4] = global_timer_ns();
        // publish the whole record at once
        uint32_t *ph = reinterpret_cast<uint32_t *>(cc.recX);
        uint32_t *pv = ph + C::PANEL_WORDS;
        uint16_t *edge = reinterpret_cast<uint16_t *>(cc.recX + 2 * C::PANEL_WORDS * 4);
        for (int e = tid; e < C::PANEL_WORDS; e += C::NTHR) {
            const int g = e / T, k = e % T;
            __stcg(ph + e, sm.Wst[(8 + g) * C::TP + k]);
            __stcg(pv + e, sm.Xst[g * C::TP + k]);
        }
        if (tid < T) {
            __stcg(edge + tid, (uint16_t)sm.val[tid + 1]);                       // top row  M(I*T, c)
            __stcg(edge + T + tid, (uint16_t)sm.val[tid * C::VP + T]);           // right column M(r, J*T+T-1)
        }
    } else {
        const int s_left = si.sbase + tri_index(nt, I, J - 1);
        const int s_below = si.sbase + tri_index(nt, I + 1, J);
        const int s_ii = si.sbase + tri_index(nt, I, I);
        const int s_jj = si.sbase + tri_index(nt, J, J);
        const int s_i1 = si.sbase + tri_index(nt, I, I + 1);
        const int s_j1 = si.sbase + tri_index(nt, J - 1, J);
        const int S = nstages(dp, p.delta);
        cc.recZ = rec_ptr<Q>(p, s_left); cc.recY = rec_ptr<Q>(p, s_below);
        cc.rowprogZ = p.rowprog + s_left; cc.colprogY = p.colprog + s_below;
        if (dp >= 2) {
            const int s_c = si.sbase + tri_index(nt, I + 1, J - 1);
            cc.recC = rec_ptr<Q>(p, s_c); cc.doneC = p.done + s_c;
        }
        if (tid == 0) {
            wait_flag_ge(p.done + s_ii, 1);
            wait_flag_ge(p.done + s_jj, 1);
            if (dp >= 3) { wait_flag_ge(p.done + s_i1, 1); wait_flag_ge(p.done + s_j1, 1); }
            if (S > 0) wait_flag_ge(p.accstage + sidx, S);
            if (tr) tr[1] = global_timer_ns();
        }
        __syncthreads();
        // static words: row words of (I,I) -> Wst[0..7], column words of (J,J) -> Xst[8..15]; the tile's own
        // words are not known yet: zero (= a valid lower bound)
        {
            const uint32_t *ph = reinterpret_cast<const uint32_t *>(rec_ptr<Q>(p, s_ii));
            const uint32_t *pv = reinterpret_cast<const uint32_t *>(rec_ptr<Q>(p, s_jj)) + C::PANEL_WORDS;
            for (int e = tid; e < C::PANEL_WORDS; e += C::NTHR) {
                const int g = e / T, k = e % T;
                sm.Wst[g * C::TP + k] = __ldcg(ph + e);
                sm.Xst[(8 + g) * C::TP + k] = __ldcg(pv + e);
            }
            for (int e = tid; e < 8 * C::TP; e += C::NTHR) { sm.Wst[8 * C::TP + e] = 0; sm.Xst[e] = 0; }
            if (dp >= 3) {
                // static operands of the late products: row panel of (I,I+1), column panel of (J-1,J)
                const uint32_t *ph1 = reinterpret_cast<const uint32_t *>(rec_ptr<Q>(p, s_i1));
                const uint32_t *pv1 = reinterpret_cast<const uint32_t *>(rec_ptr<Q>(p, s_j1)) + C::PANEL_WORDS;
                uint32_t *WI1 = panel_WI1<Q>(sm), *XJ1 = panel_XJ1<Q>(sm);
                for (int e = tid; e < C::PANEL_WORDS; e += C::NTHR) { WI1[e] = __ldcg(ph1 + e); XJ1[e] = __ldcg(pv1 + e); }
            }
        }
        // bulk maxima gathered by the PROD stages (or zero)
        if (S > 0) {
            const int16_t *accg = p.acc + (size_t)sidx * T * T;
            for (int e = tid; e < T * T; e += C::NTHR) sm.val[(e / T) * C::VP + (e % T) + 1] = __ldcg(accg + e);
        } else {
            for (int e = tid; e < T * T; e += C::NTHR) sm.val[(e / T) * C::VP + (e % T) + 1] = 0;
        }
        __syncthreads();
        if (tr && tid == 0) tr[2] = tr[3] = global_timer_ns();
        if (warp < C::NWV) close_wave<Q, false>(sm, cc, warp, lane);
        else if (warp < C::NWV + C::NMH) close_mini_helper<Q, false>(sm, cc, warp - C::NWV, lane);
        else if (warp == C::NWV + C::NMH) close_row_loader<Q>(sm, cc, lane);
        else if (warp == C::NWV + C::NMH + 1) close_col_loader<Q>(sm, cc, lane);
        else if (warp == C::NWV + C::NMH + 2) close_row_late<Q>(sm, cc, 0, lane);
        else if (warp == C::NWV + C::NMH + 3) close_col_late<Q>(sm, cc, 1, lane);
        else if (warp == C::NWV + C::NMH + 4) close_publisher<Q>(sm, cc, 1, lane);
        else if (warp == C::NWV + C::NMH + 5) close_publisher<Q>(sm, cc, 0, lane);
        else if (warp == C::NWV + C::NMH + 6) close_row_late<Q>(sm, cc, 1, lane);
        else if (warp == C::NWV + C::NMH + 7) close_col_late<Q>(sm, cc, 0, lane);
        __syncthreads();
        if (tr && tid == 0) tr[4] = global_timer_ns();
    }

    // ---- optional table block, score, completion flags (step a8) ----
    {
        const int n = si.n;
        if (p.table_out) {
            // out[(i-1)*n + (j-1)] = D(i,j) = M(i-1, j): r = i-1 <= n-1, 1 <= c <= n, c >= r+1
            for (int e = tid; e < T * T; e += C::NTHR) {
                const int a = e / T, k = e % T;
                const int r = I * T + a, c = J * T + k;
                if (r < n && c >= r + 1 && c <= n) {
                    const int v = sm.val[a * C::VP + k + 1];
                    if (p.table_dtype == RNA4R_TABLE_INT16) reinterpret_cast<int16_t *>(p.table_out)[(size_t)r * n + c - 1] = (int16_t)v;
                    else reinterpret_cast<int32_t *>(p.table_out)[(size_t)r * n + c - 1] = v;
                }
            }
        }
        if (I == 0 && J == n / T && tid == 0) {
            const int o = p.map ? p.map[seq] : seq;
            p.scores[o] = si.invalid ? -1 : (int32_t)sm.val[(n - J * T) + 1];   // M(0,n) = D(1,n)
            if (p.status) p.status[o] = si.invalid;
        }
        __syncthreads();               // orders every thread's stores before thread 0's releases (cumulative)
        if (tid == 0) {
            if (dp == 0) { st_release_gpu(cc.rowprogX, 8); st_release_gpu(cc.colprogX, 8); }
            st_release_gpu(p.done + sidx, 1);
            sm.misc[1] += 1;
            if (tr) tr[5] = global_timer_ns();
        }
    }
}

template <int Q>
__global__ void __launch_bounds__(Cfg<Q>::NTHR, Cfg<Q>::MIN_CTAS) fill_kernel(Params p)
{
    using C = Cfg<Q>;
    extern __shared__ __align__(16) uint8_t smem_raw[];
    Smem<Q> sm(smem_raw);
    const int tid = threadIdx.x;
    if (!sm.ok) __trap();                      // the host sized the launch for another shared-memory base: fail loudly
    // table R (reachable quadrant) -> shared memory, once per CTA
    {
        const uint4 *src = reinterpret_cast<const uint4 *>(p.tbl);
        uint4 *dst = reinterpret_cast<uint4 *>(sm.tbl);
        if constexpr (C::TERN || C::TBL_PITCH == (1 << C::HB)) {
            for (int e = tid; e < (C::TBL_BYTES + 15) / 16; e += C::NTHR) dst[e] = __ldg(src + e);       // the device tables are padded to 16 bytes
            if (C::TBL_BYTES < 16) for (int e = tid; e < C::TBL_BYTES; e += C::NTHR) sm.tbl[e] = p.tbl[e];
        } else {
            // padded pitch: row h of the compact table -> byte offset h * TBL_PITCH
            constexpr int ROWB = 1 << C::HB;
            if constexpr (ROWB % 4 == 0) {
                const uint32_t *s32 = reinterpret_cast<const uint32_t *>(p.tbl);
                for (int e = tid; e < ROWB * ROWB / 4; e += C::NTHR) {
                    const int h = e / (ROWB / 4), w = e % (ROWB / 4);
                    *reinterpret_cast<uint32_t *>(sm.tbl + h * C::TBL_PITCH + 4 * w) = __ldg(s32 + e);
                }
            } else {
                for (int e = tid; e < ROWB * ROWB; e += C::NTHR) sm.tbl[(e / ROWB) * C::TBL_PITCH + e % ROWB] = p.tbl[e];
            }
        }
    }
    if (tid < C::MB_COUNT) {
        const int u = tid - C::MB_STEPIN;
        mbar_init(sm.mbar + tid, (u >= 0 && u < 12) ? C::stepin_count(u) : 1);
    }
    if (tid == 0) sm.misc[1] = 0;
    __syncthreads();
    const int total = p.hdr->total;
    for (;;) {
        if (tid == 0) sm.misc[0] = atomicAdd(&p.hdr->counter, 1);
        __syncthreads();
        const int tk = sm.misc[0];
        if (tk >= total) break;
        const int4 task = p.tasks[tk];
        const SeqInfo si = p.seqinfo[task.x];
        const int I = task.y & 0xffff, J = (task.y >> 16) & 0xffff;
        if (task.z == TASK_PROD) run_prod<Q>(p, sm, si, I, J, task.w);
        else run_close<Q>(p, sm, si, task.x, I, J);
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// host side: workspace layout and enqueue
// ------------------------------------------------------------------------------------------------
// Member diagonals per product stage: longer stages mean fewer merge passes over the acc tile (they pay off on
// long folds, measured at n = 16384), shorter ones feed the closures earlier.
static inline int pick_delta(int T, const int32_t *lens, int count, int n_single)
{
    int max_n = 0;
    for (int t = 0; t < count; ++t) { const int n = lens ? lens[t] : n_single; if (n > max_n) max_n = n; }
    const int nt = max_n / T + 1;
    return nt > 192 ? 16 : nt > 128 ? 8 : 4;     // n = 16384: 18.0 ms with 8 and with 16, half the acc traffic with 16
}

struct HostPlan {
    size_t tiles, codes, tasks;
    int max_nt;
};

static inline HostPlan host_plan(int T, int delta, const int32_t *lens, int count, int n_single)
{
    HostPlan h{0, 0, 0, 1};
    for (int t = 0; t < count; ++t) {
        const int n = lens ? lens[t] : n_single;
        const int nt = n / T + 1;
        h.tiles += (size_t)nt * (nt + 1) / 2;
        h.codes += (size_t)nt * T;
        if (nt > h.max_nt) h.max_nt = nt;
        h.tasks += (size_t)nt * (nt + 1) / 2;
        for (int dp = 4; dp <= nt - 1; ++dp) h.tasks += (size_t)nstages(dp, delta) * (nt - dp);
    }
    return h;
}

struct WsLayout {
    size_t zero_bytes;   // prefix that must be zeroed before every fold
    size_t off_hdr, off_stepC, off_stepP, off_curC, off_curP, off_done, off_accstage, off_rowprog, off_colprog;
    size_t off_seqinfo, off_lens, off_map, off_tasks, off_codes, off_recs, off_acc, total;
};

static inline WsLayout ws_layout(int T, int rec_bytes, const HostPlan &h, int count)
{
    WsLayout w;
    size_t off = 0;
    w.off_hdr = off; off += 256;
    w.off_stepC = off; off += align_up((size_t)h.max_nt * 4, 256);
    w.off_stepP = off; off += align_up((size_t)h.max_nt * 4, 256);
    w.off_curC = off; off += align_up((size_t)h.max_nt * 4, 256);
    w.off_curP = off; off += align_up((size_t)h.max_nt * 4, 256);
    w.off_done = off; off += align_up(h.tiles * 4, 256);
    w.off_accstage = off; off += align_up(h.tiles * 4, 256);
    w.off_rowprog = off; off += align_up(h.tiles * 4, 256);
    w.off_colprog = off; off += align_up(h.tiles * 4, 256);
    w.off_seqinfo = off; off += align_up((size_t)count * sizeof(SeqInfo), 256);
    w.zero_bytes = off;
    w.off_lens = off; off += align_up((size_t)count * 4, 256);
    w.off_map = off; off += align_up((size_t)count * 4, 256);
    w.off_tasks = off; off += align_up(h.tasks * sizeof(int4), 256);
    w.off_codes = off; off += align_up(h.codes, 256);
    w.off_recs = off; off += align_up(h.tiles * (size_t)rec_bytes, 256);
    w.off_acc = off; off += align_up(h.tiles * (size_t)T * T * 2, 256);
    w.total = off;
    return w;
}

template <int Q>
static size_t workspace_bytes_q(int delta, const int32_t *lens, int count, int n_single)
{
    using C = Cfg<Q>;
    (void)delta;
    const HostPlan h = host_plan(C::T, 4, lens, count, n_single);      // the shortest stage span gives the most tasks: sized for it
    return ws_layout(C::T, C::REC_BYTES, h, count).total;
}

template <int Q>
static int enqueue_q(rna4r_ctx *ctx, int delta, const uint8_t *seqs, const int64_t *offsets, const int32_t *lens_host,
                     int count, int n_single, int32_t *scores, int32_t *status, void *table_out, int table_dtype, void *ws,
                     cudaStream_t st, const int32_t *map_host = nullptr)
{
    using C = Cfg<Q>;
    if (delta <= 0) delta = pick_delta(C::T, lens_host, count, n_single);
    const HostPlan h = host_plan(C::T, 4, lens_host, count, n_single);  // layout as sized by workspace_bytes_q
    const WsLayout w = ws_layout(C::T, C::REC_BYTES, h, count);
    char *base = (char *)ws;
    Params p;
    p.seqs = seqs; p.offsets = offsets; p.n_single = n_single; p.count = count; p.max_nt = h.max_nt; p.delta = delta;
    p.lens_dev = (const int32_t *)(base + w.off_lens); p.status = status;
    p.map = map_host ? (const int32_t *)(base + w.off_map) : nullptr;
    p.hdr = (PlanHdr *)(base + w.off_hdr);
    p.stepC = (int *)(base + w.off_stepC); p.stepP = (int *)(base + w.off_stepP);
    p.curC = (int *)(base + w.off_curC); p.curP = (int *)(base + w.off_curP);
    p.done = (int *)(base + w.off_done); p.accstage = (int *)(base + w.off_accstage);
    p.rowprog = (int *)(base + w.off_rowprog); p.colprog = (int *)(base + w.off_colprog);
    p.seqinfo = (SeqInfo *)(base + w.off_seqinfo);
    p.tasks = (int4 *)(base + w.off_tasks);
    p.codes = (int8_t *)(base + w.off_codes);
    p.recs = (uint8_t *)(base + w.off_recs);
    p.acc = (int16_t *)(base + w.off_acc);
    p.tbl = C::TERN ? ctx->Rt : ctx->Rc;
    p.scores = scores; p.table_out = table_out; p.table_dtype = table_dtype;
    p.trace = ctx->trace; p.trace_tiles = ctx->trace_tiles;
    p.sm_count = ctx->sm_count;

    if (ctx->tiled_blocks_per_sm == 0)     // first launch of this context (one q, one device): opt in to the large shared window
        RNA4R_CUDA(ctx, cudaFuncSetAttribute(fill_kernel<Q>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES));
    if (ctx->tiled_blocks_per_sm == 0) {
        int nb = 0;
        RNA4R_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fill_kernel<Q>, C::NTHR, C::SMEM_BYTES));
        if (nb < 1) return RNA4R_ERR_CUDA;
        ctx->tiled_blocks_per_sm = nb;
    }
    int launches = 0;
    RNA4R_CUDA(ctx, cudaMemsetAsync(ws, 0, w.zero_bytes, st));
    if (offsets)    // lens_host is consumed before this call returns (pageable memory is staged by the runtime)
        RNA4R_CUDA(ctx, cudaMemcpyAsync(base + w.off_lens, lens_host, (size_t)count * 4, cudaMemcpyHostToDevice, st));
    if (map_host)
        RNA4R_CUDA(ctx, cudaMemcpyAsync(base + w.off_map, map_host, (size_t)count * 4, cudaMemcpyHostToDevice, st));
    if (!offsets && h.max_nt <= 2048) {
        plan_single_kernel<Q><<<h.max_nt, 128, 0, st>>>(p); ++launches;          // plan + encode of a single fold: one launch
    } else {
        plan_seq_kernel<Q><<<count, 64, 0, st>>>(p); ++launches;
        plan_scan_kernel<<<1, 32, 0, st>>>(p); ++launches;
        plan_fill_kernel<Q><<<count * h.max_nt, 64, 0, st>>>(p); ++launches;
        const int maxlen = h.max_nt * C::T;
        dim3 grid((maxlen + 255) / 256, count < 65535 ? count : 65535);
        encode_kernel<Q><<<grid, 256, 0, st>>>(p); ++launches;
    }
    size_t want = h.tasks;
    int per_sm = ctx->tiled_blocks_per_sm;
    // A single fold of moderate length is bound by the closure chain, and a closure runs faster with fewer
    // neighbours on its SM (measured at n=6000: 1.98 ms with 2 CTAs/SM, 2.11 ms with 3; n=2000: 0.60 / 0.64); long folds and
    // batches are throughput-bound and take every CTA they can get (n=8000: 3.43 ms with 3, 3.48 with 2; n=16384: 18.8 / 21).
    if (count == 1 && h.max_nt <= 112 && per_sm > 2) per_sm = 2;
    // Up to n ~ 4000 no super-tile diagonal has more closures in flight than there are SMs, and a closure that has its SM
    // to itself runs 1.3x faster: one CTA per SM (n = 2000: 0.467 ms against 0.500 with two, n = 4000: 0.969 / 1.031;
    // n = 5000: 1.469 / 1.361, n = 6000: 2.15 / 1.77 -- there the products need the second CTA)
    if (count == 1 && h.max_nt <= 64) per_sm = 1;
    if (ctx->max_blocks_per_sm >= 1 && ctx->max_blocks_per_sm < per_sm) per_sm = ctx->max_blocks_per_sm;   // rna4r_set_max_blocks_per_sm
    int blocks = ctx->sm_count * per_sm;
    if ((size_t)blocks > want) blocks = (int)want;
    if (ctx->max_blocks >= 1 && blocks > ctx->max_blocks) blocks = ctx->max_blocks;
    if (blocks < 1) blocks = 1;
    if (ctx->timing) RNA4R_CUDA(ctx, cudaEventRecord(ctx->ev0, st));
    fill_kernel<Q><<<blocks, C::NTHR, C::SMEM_BYTES, st>>>(p); ++launches;
    if (ctx->timing) { RNA4R_CUDA(ctx, cudaEventRecord(ctx->ev1, st)); ctx->timing_valid = 1; }
    RNA4R_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = launches;
    return RNA4R_OK;
}

}  // namespace tiled
