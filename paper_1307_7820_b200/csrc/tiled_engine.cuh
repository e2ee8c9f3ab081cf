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
// Each (row, group) is one 32-bit word  W = M(r,gq) << SH | h << HB  and each (group, column) one
// word X = M(gq,c) << SH | v  (HB = q-1, SH = 2*HB).  Then S = W + X carries the table index in its
// low SH bits and the anchor sum above them, and  S + (Rc[idx] << SH)  is the candidate, still
// tagged with harmless low bits: one add, one mask, one byte gather, one shift-add, one max.
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
#include <cstdlib>

namespace tiled {

#ifndef RNA4R_ROLES
#define RNA4R_ROLES 2
#endif

template <int Q>
struct Cfg {
    static constexpr int T = 8 * Q;            // cells per super-tile side
    static constexpr int HB = Q - 1;           // informative bits per vector
    static constexpr int SH = 2 * HB;          // table index bits
    static constexpr uint32_t IDXMASK = (1u << SH) - 1u;
    static constexpr bool NIBBLE = (SH > 16);  // q = 10: nibble-packed table (128 KB)
    static constexpr int TBL_BYTES = NIBBLE ? (1 << SH) / 2 : (1 << SH);
    // q <= 8: the byte table sits at a shared-memory address aligned to its size, so that the gather
    // address is (S & IDXMASK) | base -- one LOP3 -- instead of mask + add
    static constexpr bool TBL_ALIGNED = (Q <= 8);
    static constexpr int TBL_ALIGN = TBL_ALIGNED ? (TBL_BYTES < 16 ? 16 : TBL_BYTES) : 16;
    static constexpr int NTHR = 4 * T;         // threads per CTA
    static constexpr int RPT = 2 * Q;          // rows per thread in the product phase
    static constexpr int TP = T + 8;           // pitch of the per-group word arrays (bank spread)
    static constexpr int VP = T + 1;           // pitch of the value array (int16): a wavefront step is conflict-free
    static constexpr int PANEL_WORDS = 8 * T;  // words in one row or column panel
    static constexpr int REC_BYTES = 2 * PANEL_WORDS * 4 + 2 * T * 2;   // PH, PV, top row, right column
    // closure wavefront: R lanes ("roles") share one column, CPW columns per warp
    static constexpr int R = RNA4R_ROLES;
    static constexpr int CPW = 32 / R;
    static constexpr int NCW = (T + CPW - 1) / CPW;      // wavefront warps (<= NTHR/32)
    static constexpr int WROWS = 16 + R + 1;             // word-array rows: 16 groups + zero guard rows
    static constexpr int ESLOTS = T + 2;                 // hand-off slots per warp boundary
    // shared-memory layout: [E | Wst | Xst | pad | tbl (aligned) | val | stg | codeR | codeC | misc]
    static constexpr int E_BYTES = 2 * (NCW > 1 ? NCW - 1 : 1) * ESLOTS * 8;
    static constexpr int W_BYTES = WROWS * TP * 4;
    static constexpr int PRE_BYTES = (E_BYTES + 2 * W_BYTES + 15) / 16 * 16;
    static constexpr int VAL_BYTES = (((T + 1) * VP + 1) * 2 + 15) / 16 * 16;
    static constexpr int STG_BYTES = 2 * 2 * PANEL_WORDS * 4;
    static constexpr int POST_BYTES = VAL_BYTES + STG_BYTES + ((2 * T + 15) / 16 * 16) + 64;
    static_assert(NCW * 32 <= NTHR || T < 32, "wavefront warps must fit the CTA");
    // dynamic shared memory needed when the dynamic window starts at shared address `base`
    static constexpr size_t smem_bytes_for(size_t base)
    {
        const size_t tbl_at = (base + PRE_BYTES + TBL_ALIGN - 1) / TBL_ALIGN * TBL_ALIGN;
        return tbl_at - base + (size_t)((TBL_BYTES + 15) / 16 * 16) + POST_BYTES;
    }
    static constexpr size_t SMEM_BYTES = smem_bytes_for(0) > smem_bytes_for(1024) ? smem_bytes_for(0) : smem_bytes_for(1024);
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
    constexpr int T = Cfg<Q>::T;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= p.count) return;
    const int n = p.offsets ? (int)(p.offsets[t + 1] - p.offsets[t]) : p.n_single;
    const int nt = n / T + 1;
    SeqInfo si;
    si.n = n; si.nt = nt; si.invalid = 0; si.pad[0] = si.pad[1] = si.pad[2] = 0;
    si.sbase = atomicAdd(&p.hdr->ntiles, nt * (nt + 1) / 2);
    si.cbase = atomicAdd(&p.hdr->ncodes, nt * T);
    p.seqinfo[t] = si;
    for (int D = 0; D < nt; ++D) {
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
    const int t = blockIdx.y;
    const SeqInfo si = p.seqinfo[t];
    const int len = si.nt * T;
    const uint8_t *src = p.seqs + (p.offsets ? p.offsets[t] : 0);
    bool bad = false;
    for (int x = blockIdx.x * blockDim.x + threadIdx.x; x < len; x += gridDim.x * blockDim.x) {
        int c = 4;
        if (x < si.n) { c = rna4r_base_code(src[x]); bad |= (c == 4); }
        p.codes[si.cbase + x] = (int8_t)c;
    }
    if (bad) atomicOr(&p.seqinfo[t].invalid, 1);
}

// ------------------------------------------------------------------------------------------------
// fill kernel
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <int Q>
struct Smem {
    using C = Cfg<Q>;
    uint2 *E;            // [2][NCW-1][ESLOTS] tagged hand-off slots between wavefront warps
    uint32_t *Wst;       // [WROWS][TP] row words:    groups 0..7 of block I (static), 8..15 of block J (own), then zero rows
    uint32_t *Xst;       // [WROWS][TP] column words: groups 0..7 of block I (own),    8..15 of block J (static), then zero rows
    uint8_t *tbl;        // compact table Rc
    uint32_t tbl_sa;     // its shared-space address (aligned to TBL_ALIGN)
    int16_t *val;        // [(T+1)][VP] values; column 0 = right column of (I,J-1), row T = top row of (I+1,J)
    uint32_t *stg;       // [2][2][PANEL_WORDS] product operands, double buffered: [buf][0]=PH, [buf][1]=PV
    int8_t *codeR;       // [T] codes of the rows
    int8_t *codeC;       // [T] codes of the columns
    int *misc;           // [16]
    bool ok;             // the layout fits the dynamic shared memory of this launch
    __device__ explicit Smem(uint8_t *base)
    {
        uint8_t *p = base;
        E = (uint2 *)p; p += C::E_BYTES;
        Wst = (uint32_t *)p; p += C::W_BYTES;
        Xst = (uint32_t *)p; p += C::W_BYTES;
        const uint32_t sa0 = smem_addr(base);
        const uint32_t tsa = (sa0 + C::PRE_BYTES + C::TBL_ALIGN - 1) / C::TBL_ALIGN * C::TBL_ALIGN;
        p = base + (tsa - sa0);
        tbl = p; tbl_sa = tsa; p += (C::TBL_BYTES + 15) / 16 * 16;
        val = (int16_t *)p; p += C::VAL_BYTES;
        stg = (uint32_t *)p; p += C::STG_BYTES;
        codeR = (int8_t *)p; p += C::T;
        codeC = (int8_t *)p; p += C::T;
        p = base + ((p - base) + 15) / 16 * 16;
        misc = (int *)p; p += 64;
        uint32_t dyn;
        asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn));
        ok = (uint32_t)(p - base) <= dyn;
    }
};

// One table gather (the unit of work of this path): rv = Rc[S & IDXMASK].
template <int Q>
__device__ __forceinline__ uint32_t tbl_gather(const Smem<Q> &sm, uint32_t S)
{
    using C = Cfg<Q>;
    if constexpr (C::NIBBLE) {
        const uint32_t idx = S & C::IDXMASK;
        const uint32_t w = reinterpret_cast<const uint32_t *>(sm.tbl)[idx >> 3];
        return (w >> ((idx & 7u) * 4u)) & 15u;
    } else if constexpr (C::TBL_ALIGNED) {
        uint32_t rv;
        const uint32_t a = (S & C::IDXMASK) | sm.tbl_sa;          // one LOP3: the table is aligned to its size
        asm("ld.shared.u8 %0, [%1];" : "=r"(rv) : "r"(a));
        return rv;
    } else {
        return sm.tbl[S & C::IDXMASK];
    }
}

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void wait_flag_ge(const int *flag, int v)
{
    while (ld_acquire_gpu(flag) < v) __nanosleep(40);
}

template <int Q>
__device__ __forceinline__ const uint8_t *rec_ptr(const Params &p, int sidx) { return p.recs + (size_t)sidx * Cfg<Q>::REC_BYTES; }

// issue the async copy of PH(I,K) and PV(K,J) into stage buffer `buf` (one 16-byte chunk per thread)
template <int Q>
__device__ __forceinline__ void load_operands_async(const Params &p, const Smem<Q> &sm, int buf, int sidx_ik, int sidx_kj)
{
    using C = Cfg<Q>;
    const int tid = threadIdx.x;
    constexpr int CH = C::PANEL_WORDS / 4;        // 16-byte chunks per panel = 2T
    uint32_t *dst = sm.stg + (size_t)buf * 2 * C::PANEL_WORDS;
    if (tid < CH) {
        cp_async16(dst + tid * 4, rec_ptr<Q>(p, sidx_ik) + (size_t)tid * 16);                               // PH of (I,K)
    } else {
        const int c = tid - CH;
        cp_async16(dst + C::PANEL_WORDS + c * 4, rec_ptr<Q>(p, sidx_kj) + (size_t)C::PANEL_WORDS * 4 + (size_t)c * 16);   // PV of (K,J)
    }
    cp_async_commit();
}

// bulk step (a4): acc[rr] = max over the 8 groups of block K, for column jj and rows rb*RPT+rr.
// acc is kept in the tagged form (value << SH | low bits); unsigned max orders by value.
template <int Q>
__device__ __forceinline__ void product_accumulate(const Smem<Q> &sm, int buf, uint32_t (&acc)[Cfg<Q>::RPT], int jj, int rb)
{
    using C = Cfg<Q>;
    const uint32_t *PH = sm.stg + (size_t)buf * 2 * C::PANEL_WORDS;
    const uint32_t *PV = PH + C::PANEL_WORDS;
#pragma unroll 2
    for (int g = 0; g < 8; ++g) {
        const uint32_t X = PV[g * C::T + jj];
        const uint32_t *wrow = PH + g * C::T + rb * C::RPT;
        uint32_t w[C::RPT];
        // the row words are warp-uniform: broadcast vector loads (16 B when RPT % 4 == 0, else 8 B)
        if constexpr (C::RPT % 4 == 0) {
#pragma unroll
            for (int r4 = 0; r4 < C::RPT / 4; ++r4) {
                const uint4 t4 = reinterpret_cast<const uint4 *>(wrow)[r4];
                w[4 * r4] = t4.x; w[4 * r4 + 1] = t4.y; w[4 * r4 + 2] = t4.z; w[4 * r4 + 3] = t4.w;
            }
        } else {
#pragma unroll
            for (int r2 = 0; r2 < C::RPT / 2; ++r2) {
                const uint2 t2 = reinterpret_cast<const uint2 *>(wrow)[r2];
                w[2 * r2] = t2.x; w[2 * r2 + 1] = t2.y;
            }
        }
#pragma unroll
        for (int rr = 0; rr < C::RPT; ++rr) {
            const uint32_t S = w[rr] + X;
            const uint32_t rv = tbl_gather<Q>(sm, S);
            const uint32_t cand = S + (rv << C::SH);
            acc[rr] = max(acc[rr], cand);
        }
    }
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
    const int jj = tid % C::T, rb = tid / C::T;
    uint32_t acc[C::RPT];
#pragma unroll
    for (int rr = 0; rr < C::RPT; ++rr) acc[rr] = 0;

    // K sequence: for m = lo..hi: K = I+m, then K = J-m (if different)
    const int nk_max = 2 * (hi - lo + 1);
    int issued = 0, computed = 0;
    auto kth = [&](int e) -> int {           // e-th block of the sequence, or -1 for the duplicate
        const int m = lo + (e >> 1);
        const int K = (e & 1) ? (J - m) : (I + m);
        if ((e & 1) && (J - m == I + m)) return -1;
        return K;
    };
    // software pipeline: operands of element e+1 are in flight while element e is computed
    int e_next = 0;
    auto issue_next = [&]() -> bool {
        while (e_next < nk_max) {
            const int K = kth(e_next++);
            if (K < 0) continue;
            const int s_ik = si.sbase + tri_index(nt, I, K), s_kj = si.sbase + tri_index(nt, K, J);
            if (tid == 0) { wait_flag_ge(p.done + s_ik, 1); wait_flag_ge(p.done + s_kj, 1); }
            __syncthreads();
            load_operands_async<Q>(p, sm, issued & 1, s_ik, s_kj);
            ++issued;
            return true;
        }
        return false;
    };
    issue_next();
    while (computed < issued) {
        const bool more = issue_next();
        if (more) cp_async_wait<1>(); else cp_async_wait<0>();
        __syncthreads();
        product_accumulate<Q>(sm, computed & 1, acc, jj, rb);
        ++computed;
        __syncthreads();     // the buffer may be refilled by the next issue
    }
    // merge with earlier stages (they ran at earlier steps and own acc until their release)
    int16_t *accg = p.acc + (size_t)sidx * C::T * C::T;
    if (s != S - 1) {
        if (tid == 0) wait_flag_ge(p.accstage + sidx, S - 1 - s);
        __syncthreads();
#pragma unroll
        for (int rr = 0; rr < C::RPT; ++rr) {
            const int prev = __ldcg(accg + (size_t)(rb * C::RPT + rr) * C::T + jj);
            acc[rr] = max(acc[rr], (uint32_t)prev << C::SH);
        }
    }
#pragma unroll
    for (int rr = 0; rr < C::RPT; ++rr)
        __stcg(accg + (size_t)(rb * C::RPT + rr) * C::T + jj, (int16_t)(acc[rr] >> C::SH));
    __threadfence();
    __syncthreads();
    if (tid == 0) st_release_gpu(p.accstage + sidx, S - s);
}

// ------------------------------------------------------------------------------------------------
// closure of one super-tile (steps a3, a5, a6, a7 inside the CTA): a continuous skewed wavefront
//
// Local coordinates: rows a = 0..T-1 (a = T-1 is the bottom row), columns c = 0..T-1.  Lane <-> column:
// the lane that owns column c walks it bottom-up, one cell per step, one row below its left
// neighbour: at step k it is on row a = T-1-k+c, so all cells of one anti-diagonal
// are computed in the same step and the whole tile takes 2T-1 steps, with no barrier between them.
// CPW = 32/R columns per warp; the R lanes ("roles") of a column hold identical wavefront state and
// split the table lookups of the step.  Neighbouring warps are coupled by tagged hand-off slots in
// shared memory (value + row word of the warp's last two columns), polled by the consumer.
//
// Critical-path split.  Of all candidates of cell (a,c) only two depend on the previous step:
//   left  = v(a,c-1)  (tail split t = c-1: M(r,c-1) + M(c-1,c), M(c-1,c) = 0)   -- one shuffle
//   below = v(a+1,c)  (head split t = r+1: M(r,r+1) + M(r+1,c), M(r,r+1) = 0)   -- own register.
// Everything else of cell (a-1,c) -- the bulk maximum, b + D(i+1,j-1) and every
// lookup over rows >= a+1 and columns <= c-2 -- is computed during step k ("OLDX") and only enters
// v(a-1,c) at step k+1.  So the dependent chain of a step is  shuffle -> max.
//
// Lookups of one step, target cell (a-1,c).  With the word arrays indexed by z = 0..15 (z < 8: group
// z of block I, z >= 8: group z-8 of block J) the groups to look up are one contiguous range
// z = zL..zR,  zL = floor((a+1)/Q),  zR = 8 + floor((c-2)/Q):
//   z = zL  head special: the running column word Xp (rows >= a+1 of the lane's own column) with the
//           row word of (I,I)                                 -- the paper's head residual loop
//   z = zR  tail special: the row word of row a-1 through column c-2 (from lane c-2, by shuffle) with
//           the column word of (J,J)                          -- the paper's tail residual loop
//   zL < z < zR  interior: both words complete, read from shared memory (full groups)
// (PAPER.md:145-155 residual loops as masked lookups: DESIGN.md 4.3).  Words that are not complete yet
// are zero (the arrays are cleared per tile), and a zero word only yields a valid lower bound, so the
// walk over the interior may overshoot without harm; its trip count is warp-uniform.
// DIAG (I == J): row and column words are both the tile's own; only z < 8 is used (zR = floor((c-2)/Q)),
// plus the merged lookup (row word through c-2, Xp) when zL == zR; cells with c-a <= 1 are 0.
// ------------------------------------------------------------------------------------------------
constexpr uint32_t E_TAG = 0x5a5a0000u;

__device__ __forceinline__ uint2 lds_volatile_u2(const uint2 *p)
{
    uint2 r;
    asm volatile("ld.volatile.shared.v2.u32 {%0, %1}, [%2];" : "=r"(r.x), "=r"(r.y) : "r"(smem_addr(p)) : "memory");
    return r;
}
__device__ __forceinline__ void sts_volatile_u2(uint2 *p, uint32_t x, uint32_t y)
{
    asm volatile("st.volatile.shared.v2.u32 [%0], {%1, %2};" ::"r"(smem_addr(p)), "r"(x), "r"(y) : "memory");
}

template <int Q>
__device__ __forceinline__ uint32_t lookup_tagged(const Smem<Q> &sm, uint32_t W, uint32_t X)
{
    const uint32_t S = W + X;
    return S + (tbl_gather<Q>(sm, S) << Cfg<Q>::SH);      // (value << SH) | harmless low bits
}

template <int Q, bool DIAG>
__device__ __forceinline__ void wave_closure(const Smem<Q> &sm, int cw, int lane)
{
    using C = Cfg<Q>;
    constexpr int T = C::T, TP = C::TP, VP = C::VP, SH = C::SH, HB = C::HB, R = C::R, CPW = C::CPW, NCW = C::NCW;
    constexpr uint32_t FULL = 0xffffffffu;
    constexpr int OFFQ = 64 * Q;                         // keeps the operand of the constant divisions positive
    const int j = lane % CPW, rho = lane / CPW;
    const int c = cw * CPW + j;                          // my column (>= T: idle lane, never stores)
    const bool colok = c < T;
    const int b = c % Q, B = c / Q;
    const int zR = (DIAG ? 0 : 8) + (c >= 2 ? (c - 2) / Q : 0);
    const uint32_t w2keep = (c >= 2) ? FULL : 0u;
    const int want = 3 - (int)sm.codeC[colok ? c : 0];   // row code that pairs with my column (code 4 -> never)
    const int B0c = sm.val[T * VP + c + 1];              // bottom edge M((I+1)T, c)
    const uint32_t XR = DIAG ? 0u : sm.Xst[zR * TP + c]; // static column word of (J,J) for the tail special
    const int shb = HB + (b > 0 ? b - 1 : 0);            // position of my horizontal difference bit
    uint2 *E1 = sm.E + (size_t)(2 * cw) * C::ESLOTS, *E2 = E1 + C::ESLOTS;             // slots I produce
    const uint2 *P1 = sm.E + (size_t)(2 * (cw > 0 ? cw - 1 : 0)) * C::ESLOTS, *P2 = P1 + C::ESLOTS;   // slots I consume
    const int k0 = cw * CPW - 1;                         // pre-step of my first column
    const int kstart = DIAG ? max(k0, T) : k0;
    const int kend = min(T - 1 + (cw + 1) * CPW - 1, 2 * T - 2);
    const bool r0 = (rho == 0);

    int vout = 0, vprev = 0, oldx = 0;
    uint32_t wout = 0, Xp = 0;
#pragma unroll 1
    for (int k = kstart; k <= kend; ++k) {
        const int a = T - 1 - k + c;
        const int d = k - (T - 1);                       // c - a, the same for every lane
        // ---- receive from the left
        int Lv = __shfl_up_sync(FULL, vout, 1, CPW);                // v(a, c-1)
        uint32_t Lw = __shfl_up_sync(FULL, wout, 1, CPW);           // row a   through column c-1
        uint32_t Lw2 = __shfl_up_sync(FULL, wout, 2, CPW);          // row a-1 through column c-2
        if (cw == 0) {
            if (j == 0) Lv = sm.val[a * VP];                        // left edge (a = T: the corner)
            if (j < 2) Lw2 = 0;
        } else {
            const int a0 = T - 1 - k + cw * CPW;                    // row of my first column, warp-uniform
            uint2 e1 = make_uint2(0u, 0u), e2 = make_uint2(0u, 0u);
            if (!(DIAG && k == T)) {                                // DIAG: step T-1 is not run, its cells are 0
                if (a0 >= 0)
                    for (;;) { e1 = lds_volatile_u2(P1 + a0); if (__all_sync(FULL, (e1.x & 0xffff0000u) == E_TAG)) break; }
                if (a0 >= 1)
                    for (;;) { e2 = lds_volatile_u2(P2 + a0 - 1); if (__all_sync(FULL, (e2.x & 0xffff0000u) == E_TAG)) break; }
            }
            if (j == 0) { Lv = (int)(e1.x & 0xffffu); Lw = e1.y; Lw2 = e2.y; }
            if (j == 1) Lw2 = e1.y;
        }
        // ---- the cell (a3 init + a5 fresh splits)
        int v = max(max(oldx, vprev), Lv);
        if (a == T) v = B0c;                                        // pre-step: the cell below the tile
        if (DIAG && d <= 1) v = 0;                                  // D(i,i) = D(i,i-1) = 0
        const bool live = colok && (unsigned)a < (unsigned)T;
        if (live && r0) sm.val[a * VP + c + 1] = (int16_t)v;
        // ---- step a6, horizontal: my row word = neighbour's word | my difference bit
        const uint32_t wme = (b == 0) ? ((uint32_t)v << SH) : (Lw | ((uint32_t)(v - Lv) << shb));
        if (live && r0 && b == Q - 1) {
            sm.Wst[(8 + B) * TP + a] = wme;
            if (DIAG) sm.Wst[B * TP + a] = wme;
        }
        if (cw < NCW - 1 && r0 && colok && (unsigned)a <= (unsigned)T) {
            if (j == CPW - 1) sts_volatile_u2(E1 + a, E_TAG | (uint32_t)(v & 0xffff), wme);
            if (j == CPW - 2) sts_volatile_u2(E2 + a, E_TAG, wme);
        }
        // ---- OLDX of the next cell (a-1, c)
        int o = sm.val[(a - 1) * VP + c + 1];                       // bulk maximum
        if ((int)sm.codeR[a - 1] == want) o = max(o, Lv + 1);       // b(S_i,S_j) + D(i+1,j-1)
        const int zL = min((int)((unsigned)(a + 1 + OFFQ) / Q) - 64, 7);   // floor((a+1)/Q); 7 when no row of the tile is below
        const int fl = (int)((unsigned)(d - 3 + OFFQ) / Q) - 64;    // floor((d-3)/Q), warp-uniform
        // warp-uniform upper bound of the interior count zR-zL-1: floor differences give 8+fl; one more because
        // zR is one too high for columns 0,1 (no tail group) and zL is clamped on the bottom row
        const int nint = min(DIAG ? fl : 9 + fl, DIAG ? 6 : 14);
        const int nit = nint > 0 ? (nint + R - 1) / R : 0;
        const uint32_t Wh = sm.Wst[zL * TP + a - 1];
        const uint32_t Xt = DIAG ? sm.Xst[zR * TP + c] : XR;
        const uint32_t Lw2m = Lw2 & w2keep;
        uint32_t best;
        if (R == 1) {
            best = max(lookup_tagged<Q>(sm, Wh, Xp), lookup_tagged<Q>(sm, Lw2m, Xt));
        } else {
            const uint32_t W0 = (rho == 0) ? Wh : (rho == 1 ? Lw2m : 0u);
            const uint32_t X0 = (rho == 0) ? Xp : (rho == 1 ? Xt : 0u);
            best = lookup_tagged<Q>(sm, W0, X0);
        }
        if (DIAG) best = max(best, lookup_tagged<Q>(sm, (zL == zR) ? Lw2m : 0u, Xp));
        {
            const uint32_t *pw = sm.Wst + (zL + 1 + rho) * TP + a - 1;
            const uint32_t *px = sm.Xst + (zL + 1 + rho) * TP + c;
            constexpr int NITMAX = ((DIAG ? 6 : 14) + R - 1) / R;
#pragma unroll
            for (int i = 0; i < NITMAX; ++i) {
                if (i < nit) best = max(best, lookup_tagged<Q>(sm, pw[i * R * TP], px[i * R * TP]));
            }
        }
        if (R >= 2) best = max(best, __shfl_xor_sync(FULL, best, CPW));
        if (R >= 4) best = max(best, __shfl_xor_sync(FULL, best, 2 * CPW));
        oldx = max(o, (int)(best >> SH));
        // ---- step a6, vertical: the column word now starts at row a
        const int am = (int)((unsigned)(a + OFFQ) % Q);
        if (a >= T) {
            Xp = 0;                                                 // nothing of my column is known below the tile
        } else {
            Xp = (am == Q - 1) ? ((uint32_t)v << SH)
                               : ((Xp & C::IDXMASK) | ((uint32_t)(v - vprev) << am) | ((uint32_t)v << SH));
            if (live && r0 && am == 0) sm.Xst[(a / Q) * TP + c] = Xp;
        }
        vprev = v; vout = v; wout = wme;
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
    unsigned long long *tr = (p.trace && sidx < p.trace_tiles) ? p.trace + (size_t)sidx * 8 : nullptr;
    if (tr && tid == 0) { tr[0] = global_timer_ns(); tr[6] = ((unsigned long long)I << 32) | (unsigned)J; }

    // codes of the rows r = I*T + a (base S[r]) and of the columns c = J*T + jj (base S[c-1])
    if (tid < T) {
        sm.codeR[tid] = p.codes[si.cbase + I * T + tid];
        const int c = J * T + tid;
        sm.codeC[tid] = (c >= 1) ? p.codes[si.cbase + c - 1] : (int8_t)4;
    }

    const int warp = tid >> 5, lane = tid & 31;
    // hand-off slots of the wavefront warps: empty
    for (int e = tid; e < C::E_BYTES / 8; e += C::NTHR) sm.E[e] = make_uint2(0u, 0u);
    if (dp == 0) {
        // diagonal super-tile: everything starts from zero
        for (int e = tid; e < C::VAL_BYTES / 4; e += C::NTHR) reinterpret_cast<uint32_t *>(sm.val)[e] = 0;
        for (int e = tid; e < C::WROWS * C::TP; e += C::NTHR) { sm.Wst[e] = 0; sm.Xst[e] = 0; }
        __syncthreads();
        if (warp < C::NCW) wave_closure<Q, true>(sm, warp, lane);
        __syncthreads();
    } else {
        const int s_left = si.sbase + tri_index(nt, I, J - 1);
        const int s_below = si.sbase + tri_index(nt, I + 1, J);
        const int s_ii = si.sbase + tri_index(nt, I, I);
        const int s_jj = si.sbase + tri_index(nt, J, J);
        const int S = nstages(dp, p.delta);
        if (tid == 0) {
            wait_flag_ge(p.done + s_left, 1);
            wait_flag_ge(p.done + s_below, 1);
            wait_flag_ge(p.done + s_ii, 1);
            wait_flag_ge(p.done + s_jj, 1);
            if (S > 0) wait_flag_ge(p.accstage + sidx, S);
            if (tr) tr[1] = global_timer_ns();
        }
        __syncthreads();
        // static words: row words of (I,I) -> Wst[0..7], column words of (J,J) -> Xst[8..15]
        {
            const uint32_t *ph = reinterpret_cast<const uint32_t *>(rec_ptr<Q>(p, s_ii));
            const uint32_t *pv = reinterpret_cast<const uint32_t *>(rec_ptr<Q>(p, s_jj)) + C::PANEL_WORDS;
            for (int e = tid; e < C::PANEL_WORDS; e += C::NTHR) {
                const int g = e / T, k = e % T;
                sm.Wst[g * C::TP + k] = __ldcg(ph + e);
                sm.Xst[(8 + g) * C::TP + k] = __ldcg(pv + e);
            }
            // the tile's own words are not known yet: zero (= a valid lower bound); zero guard rows
            for (int e = tid; e < (C::WROWS - 8) * C::TP; e += C::NTHR) sm.Wst[8 * C::TP + e] = 0;
            for (int e = tid; e < 8 * C::TP; e += C::NTHR) sm.Xst[e] = 0;
            for (int e = tid; e < (C::WROWS - 16) * C::TP; e += C::NTHR) sm.Xst[16 * C::TP + e] = 0;
        }
        // bulk maxima gathered by the PROD stages (or zero)
        if (S > 0) {
            const int16_t *accg = p.acc + (size_t)sidx * T * T;
            for (int e = tid; e < T * T; e += C::NTHR) sm.val[(e / T) * C::VP + (e % T) + 1] = __ldcg(accg + e);
        } else {
            for (int e = tid; e < T * T; e += C::NTHR) sm.val[(e / T) * C::VP + (e % T) + 1] = 0;
        }
        // neighbours' edges: right column of (I,J-1) -> val[a][0]; top row of (I+1,J) -> val[T][jj+1];
        // corner M((I+1)T, JT-1) = top row of (I+1,J-1) at its last column (0 if that tile is below the diagonal)
        {
            const uint16_t *eleft = reinterpret_cast<const uint16_t *>(rec_ptr<Q>(p, s_left) + 2 * C::PANEL_WORDS * 4);
            const uint16_t *ebelow = reinterpret_cast<const uint16_t *>(rec_ptr<Q>(p, s_below) + 2 * C::PANEL_WORDS * 4);
            if (tid < T) {
                sm.val[tid * C::VP] = (int16_t)__ldcg(eleft + T + tid);          // right column
                sm.val[T * C::VP + tid + 1] = (int16_t)__ldcg(ebelow + tid);     // top row
            }
            if (tid == T) {
                int corner = 0;
                if (dp >= 2) {
                    const uint16_t *ec = reinterpret_cast<const uint16_t *>(
                        rec_ptr<Q>(p, si.sbase + tri_index(nt, I + 1, J - 1)) + 2 * C::PANEL_WORDS * 4);
                    corner = __ldcg(ec + T - 1);
                }
                sm.val[T * C::VP] = (int16_t)corner;
            }
        }
        __syncthreads();
        if (tr && tid == 0) tr[2] = global_timer_ns();
        // late products: the middle blocks whose panels were only finished on the previous step
        if (dp >= 2) {
            const int jj = tid % T, rb = tid / T;
            uint32_t acc[C::RPT];
#pragma unroll
            for (int rr = 0; rr < C::RPT; ++rr) acc[rr] = 0;
            const int K0 = I + 1, K1 = J - 1;
            load_operands_async<Q>(p, sm, 0, si.sbase + tri_index(nt, I, K0), si.sbase + tri_index(nt, K0, J));
            if (K1 != K0) {
                load_operands_async<Q>(p, sm, 1, si.sbase + tri_index(nt, I, K1), si.sbase + tri_index(nt, K1, J));
                cp_async_wait<1>();
            } else {
                cp_async_wait<0>();
            }
            __syncthreads();
            product_accumulate<Q>(sm, 0, acc, jj, rb);
            if (K1 != K0) {
                cp_async_wait<0>();
                __syncthreads();
                product_accumulate<Q>(sm, 1, acc, jj, rb);
            }
#pragma unroll
            for (int rr = 0; rr < C::RPT; ++rr) {
                int16_t *cell = sm.val + (rb * C::RPT + rr) * C::VP + jj + 1;
                *cell = (int16_t)max((int)*cell, (int)(acc[rr] >> C::SH));
            }
            __syncthreads();
        }
        if (tr && tid == 0) tr[3] = global_timer_ns();
        if (warp < C::NCW) wave_closure<Q, false>(sm, warp, lane);
        __syncthreads();
    }
    if (tr && tid == 0) tr[4] = global_timer_ns();

    // ---- publish: row panel, column panel, edges (step a6 output), optional table block, score ----
    {
        uint8_t *rec = const_cast<uint8_t *>(rec_ptr<Q>(p, sidx));
        uint32_t *ph = reinterpret_cast<uint32_t *>(rec);
        uint32_t *pv = ph + C::PANEL_WORDS;
        uint16_t *edge = reinterpret_cast<uint16_t *>(rec + 2 * C::PANEL_WORDS * 4);
        for (int e = tid; e < C::PANEL_WORDS; e += C::NTHR) {
            const int g = e / T, k = e % T;
            __stcg(ph + e, sm.Wst[(8 + g) * C::TP + k]);
            __stcg(pv + e, sm.Xst[g * C::TP + k]);
        }
        if (tid < T) {
            __stcg(edge + tid, (uint16_t)sm.val[tid + 1]);                       // top row  M(I*T, c)
            __stcg(edge + T + tid, (uint16_t)sm.val[tid * C::VP + T]);           // right column M(r, J*T+T-1)
        }
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
        if (I == 0 && J == n / T && tid == 0)
            p.scores[seq] = si.invalid ? -1 : (int32_t)sm.val[(n - J * T) + 1];   // M(0,n) = D(1,n)
        __threadfence();
        __syncthreads();
        if (tid == 0) { st_release_gpu(p.done + sidx, 1); if (tr) tr[5] = global_timer_ns(); }
    }
}

template <int Q>
__global__ void __launch_bounds__(Cfg<Q>::NTHR) fill_kernel(Params p)
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
        for (int e = tid; e < C::TBL_BYTES / 16; e += C::NTHR) dst[e] = __ldg(src + e);
        if (C::TBL_BYTES < 16) for (int e = tid; e < C::TBL_BYTES; e += C::NTHR) sm.tbl[e] = p.tbl[e];
    }
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
    size_t off_hdr, off_stepC, off_stepP, off_curC, off_curP, off_done, off_accstage;
    size_t off_seqinfo, off_tasks, off_codes, off_recs, off_acc, total;
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
    w.zero_bytes = off;
    w.off_seqinfo = off; off += align_up((size_t)count * sizeof(SeqInfo), 256);
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
    const HostPlan h = host_plan(C::T, delta, lens, count, n_single);
    return ws_layout(C::T, C::REC_BYTES, h, count).total;
}

template <int Q>
static int enqueue_q(rna4r_ctx *ctx, int delta, const uint8_t *seqs, const int64_t *offsets, const int32_t *lens_host,
                     int count, int n_single, int32_t *scores, void *table_out, int table_dtype, void *ws, cudaStream_t st)
{
    using C = Cfg<Q>;
    const HostPlan h = host_plan(C::T, delta, lens_host, count, n_single);
    const WsLayout w = ws_layout(C::T, C::REC_BYTES, h, count);
    char *base = (char *)ws;
    Params p;
    p.seqs = seqs; p.offsets = offsets; p.n_single = n_single; p.count = count; p.max_nt = h.max_nt; p.delta = delta;
    p.hdr = (PlanHdr *)(base + w.off_hdr);
    p.stepC = (int *)(base + w.off_stepC); p.stepP = (int *)(base + w.off_stepP);
    p.curC = (int *)(base + w.off_curC); p.curP = (int *)(base + w.off_curP);
    p.done = (int *)(base + w.off_done); p.accstage = (int *)(base + w.off_accstage);
    p.seqinfo = (SeqInfo *)(base + w.off_seqinfo);
    p.tasks = (int4 *)(base + w.off_tasks);
    p.codes = (int8_t *)(base + w.off_codes);
    p.recs = (uint8_t *)(base + w.off_recs);
    p.acc = (int16_t *)(base + w.off_acc);
    p.tbl = C::NIBBLE ? ctx->Rc4 : ctx->Rc;
    p.scores = scores; p.table_out = table_out; p.table_dtype = table_dtype;
    p.trace = ctx->trace; p.trace_tiles = ctx->trace_tiles;

    static bool attr_set = false;
    if (!attr_set) {
        RNA4R_CUDA(ctx, cudaFuncSetAttribute(fill_kernel<Q>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES));
        attr_set = true;
    }
    if (ctx->tiled_blocks_per_sm == 0) {
        int nb = 0;
        RNA4R_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fill_kernel<Q>, C::NTHR, C::SMEM_BYTES));
        if (nb < 1) return RNA4R_ERR_CUDA;
        ctx->tiled_blocks_per_sm = nb;
    }
    int launches = 0;
    RNA4R_CUDA(ctx, cudaMemsetAsync(ws, 0, w.zero_bytes, st));
    plan_seq_kernel<Q><<<(count + 127) / 128, 128, 0, st>>>(p); ++launches;
    plan_scan_kernel<<<1, 32, 0, st>>>(p); ++launches;
    plan_fill_kernel<Q><<<count * h.max_nt, 64, 0, st>>>(p); ++launches;
    {
        const int maxlen = h.max_nt * C::T;
        dim3 grid((maxlen + 255) / 256, count);
        encode_kernel<Q><<<grid, 256, 0, st>>>(p); ++launches;
    }
    size_t want = h.tasks;
    int per_sm = ctx->tiled_blocks_per_sm;
    if (const char *e = getenv("RNA4R_BLOCKS_PER_SM")) { const int v = atoi(e); if (v >= 1 && v < per_sm) per_sm = v; }   // tuning knob
    int blocks = ctx->sm_count * per_sm;
    if ((size_t)blocks > want) blocks = (int)want;
    if (blocks < 1) blocks = 1;
    if (ctx->timing) RNA4R_CUDA(ctx, cudaEventRecord(ctx->ev0, st));
    fill_kernel<Q><<<blocks, C::NTHR, C::SMEM_BYTES, st>>>(p); ++launches;
    if (ctx->timing) { RNA4R_CUDA(ctx, cudaEventRecord(ctx->ev1, st)); ctx->timing_valid = 1; }
    RNA4R_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = launches;
    return RNA4R_OK;
}

}  // namespace tiled
