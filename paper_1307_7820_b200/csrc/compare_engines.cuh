// compare_engines.cuh -- two comparison engines: what each B200 choice of the tiled engine buys.
//
// RNA4R_ENGINE_PAPER_TILE -- the paper's own CUDA design, section 5.3, as literally as the text
//   allows: "We group cells together into tiles, where each tile is a composite of q x q cells.  The tiles along a
//   diagonal can be computed independent of each other.  Each tile is assigned to a block of threads" (one launch per
//   tile-diagonal: the synchronisation of PAPER.md:242); "after all the entries of the tile are computed, only the
//   horizontal and vertical differences are stored" (plus one anchor per vector, reading g21); "the horizontal
//   difference vectors of the rows of a tile are stored in contiguous memory locations and the tiles are stored in
//   row-major order.  The vertical difference vectors of the columns of a tile are stored together and the tiles are
//   grouped in column-major order"; "when each thread retrieves one vector, the block of threads
//   accesses contiguous memory locations".  R (2^q x 2^q bytes) stays in global memory
//   behind the read-only cache.  The residual cells are plain Nussinov steps.  Any q in 2..12.
//
// RNA4R_ENGINE_MAXPLUS -- no Four-Russians table at all: eq. (1) as a blocked max-plus closure on
//   int16 values, 32 x 32 tiles, one launch per tile-diagonal, the inner max over a middle tile as DPX
//   VIADDMNMX.S16x2 (two cells per instruction).  SURVEY.md section 7: "keep a direct max-plus tile kernel as the
//   ncu-evidenced comparison".  q is ignored.
//
// Coordinates as in tiled_engine.cuh: M(r,c) = D(r+1,c), r,c in [0,n]; group / block index of a coordinate x is x / q
// (x / 32); M(r,c) = 0 for c <= r+1.
#pragma once
#include "common.cuh"

namespace cmpeng {

struct Hdr { int invalid; int pad[63]; };

// bases -> codes[0 .. len) (4 = padding); `offset` as in diag_encode_kernel
__global__ void encode_kernel(const uint8_t *__restrict__ seq, const int64_t *__restrict__ offset, int n, int len,
                              int8_t *__restrict__ codes, Hdr *hdr)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= len) return;
    int64_t start = 0;
    bool readable = true;
    if (offset) {
        start = offset[0];
        if (offset[1] - start != (int64_t)n) { readable = false; if (t == 0) atomicOr(&hdr->invalid, RNA4R_STATUS_BAD_OFFSETS); }
    }
    int c = 4;
    if (t < n && readable) { c = rna4r_base_code(seq[start + t]); if (c == 4) atomicOr(&hdr->invalid, RNA4R_STATUS_BAD_BASE); }
    codes[t] = (int8_t)c;
}

__global__ void finish_kernel(const Hdr *hdr, int32_t *score, int32_t *status, int n)
{
    if (hdr->invalid) *score = -1;
    else if (n < 2) *score = 0;
    if (status) *status = hdr->invalid;
}

template <bool I16>
__device__ __forceinline__ void store_cell(void *table_out, int n, int r, int c, int v)
{
    if (table_out && r < n && c >= r + 1 && c <= n) {
        if (I16) reinterpret_cast<int16_t *>(table_out)[(size_t)r * n + c - 1] = (int16_t)v;
        else reinterpret_cast<int32_t *>(table_out)[(size_t)r * n + c - 1] = v;
    }
}

// ====================================================================================================================
// RNA4R_ENGINE_PAPER_TILE
// ====================================================================================================================
struct PtWs {
    Hdr *hdr;
    int8_t *codes;      // [NB*q + 1]
    uint32_t *H;        // [(A*NB + g)*q + a]: anchor M(Aq+a, gq) << 16 | horizontal difference bits (bit p: p-th cell of the run)
    uint32_t *V;        // [(B*NB + g)*q + y]: anchor M(gq, Bq+y) << 16 | vertical difference bits
    size_t bytes;
};
static inline PtWs pt_layout(void *base, int n, int q)
{
    PtWs w;
    char *p = (char *)base;
    const size_t NB = (size_t)n / q + 1;
    size_t off = 0;
    w.hdr = (Hdr *)(p + off); off += 256;
    w.codes = (int8_t *)(p + off); off += align_up(NB * q + 16, 256);
    w.H = (uint32_t *)(p + off); off += align_up(NB * NB * q * 4, 256);
    w.V = (uint32_t *)(p + off); off += align_up(NB * NB * q * 4, 256);
    w.bytes = off;
    return w;
}

constexpr int PT_MAXQ = 12;

// one block <-> tile (A, A+D); thread (a,y) <-> cell (Aq+a, (A+D)q+y)
template <bool I16>
__global__ void pt_tile_kernel(int n, int q, int D, int NB, const int8_t *__restrict__ codes, const uint8_t *__restrict__ R,
                               uint32_t *__restrict__ H, uint32_t *__restrict__ V, const Hdr *hdr, int32_t *score, void *table_out)
{
    __shared__ int val[PT_MAXQ][PT_MAXQ + 1], Pd[PT_MAXQ][PT_MAXQ + 1], Qd[PT_MAXQ][PT_MAXQ + 1];
    __shared__ int Lcol[PT_MAXQ + 1], Brow[PT_MAXQ + 1];
    __shared__ uint32_t hw[PT_MAXQ], vw[PT_MAXQ];
    const int tid = threadIdx.x, a = tid / q, y = tid % q;
    const int A = blockIdx.x, B = A + D;
    const int r = A * q + a, c = B * q + y;
    const int N = 1 << q;
    if (D > 0) {
        // the neighbours are only known as differences: rebuild what the residual loops read
        if (tid < q) {
            const uint32_t w = H[((size_t)A * NB + A) * q + tid];                 // row tid of the diagonal tile (A,A)
            for (int j = 0; j < q; ++j) Pd[tid][j] = (int)(w >> 16) + __popc(w & ((2u << j) - 1u) & 0xffffu);
            const uint32_t wl = H[((size_t)A * NB + (B - 1)) * q + tid];          // row tid of the left tile: its last cell
            Lcol[tid] = (int)(wl >> 16) + __popc(wl & 0xffffu);
            Brow[tid] = (int)(V[((size_t)B * NB + (A + 1)) * q + tid] >> 16);     // top row of the tile below
            if (tid == 0) Lcol[q] = (A + 1 <= B - 1) ? (int)(V[((size_t)(B - 1) * NB + (A + 1)) * q + (q - 1)] >> 16) : 0;
        } else if (tid < 2 * q) {
            const int yy = tid - q;
            const uint32_t w = V[((size_t)B * NB + B) * q + yy];                  // column yy of the diagonal tile (B,B)
            for (int j = 0; j < q; ++j) Qd[j][yy] = (int)(w >> 16) - __popc(w & ((2u << j) - 1u) & 0xffffu);
        }
    }
    __syncthreads();
    // all groups in between (Alg. 1 lines 15-19; "each thread retrieves one vector")
    int best = 0;
    for (int g = A + 1; g <= B - 1; ++g) {
        if (tid < q) hw[tid] = H[((size_t)A * NB + g) * q + tid];
        else if (tid < 2 * q) vw[tid - q] = V[((size_t)B * NB + g) * q + (tid - q)];
        __syncthreads();
        const uint32_t h = hw[a], v = vw[y];
        best = max(best, (int)(h >> 16) + (int)(v >> 16) + (int)__ldg(R + (size_t)(h & 0xffffu) * N + (v & 0xffffu)));   // eq. (3)
        __syncthreads();
    }
    // the tile itself: 2q-1 anti-diagonals, residual cells by plain steps
    const int ca = codes[r], cc = (c >= 1) ? codes[c - 1] : 4;
    for (int s = 0; s <= 2 * q - 2; ++s) {
        if ((q - 1 - a) + y == s) {
            int v;
            if (D == 0) {
                v = 0;
                if (y > a + 1) {
                    v = val[a + 1][y - 1] + rna4r_pair(ca, cc);
                    for (int t = a + 1; t < y; ++t) v = max(v, val[a][t] + val[t][y]);
                }
            } else {
                const int dl = (a < q - 1) ? (y > 0 ? val[a + 1][y - 1] : Lcol[a + 1]) : (y > 0 ? Brow[y - 1] : Lcol[q]);
                v = max(best, dl + rna4r_pair(ca, cc));                            // D(i+1,j-1) + b(S_i,S_j)
                for (int t = a + 1; t < q; ++t) v = max(v, Pd[a][t] + val[t][y]);  // first group (Alg. 1 lines 9-11)
                for (int t = 0; t < y; ++t) v = max(v, val[a][t] + Qd[t][y]);      // last group (Alg. 1 lines 12-14)
            }
            val[a][y] = v;
        }
        __syncthreads();
    }
    // "only the horizontal and vertical differences are stored"
    if (tid < q) {
        uint32_t bits = 0;
        for (int j = 1; j < q; ++j) bits |= (uint32_t)(val[tid][j] - val[tid][j - 1]) << j;
        H[((size_t)A * NB + B) * q + tid] = ((uint32_t)val[tid][0] << 16) | bits;
    } else if (tid < 2 * q) {
        const int yy = tid - q;
        uint32_t bits = 0;
        for (int j = 1; j < q; ++j) bits |= (uint32_t)(val[j - 1][yy] - val[j][yy]) << j;
        V[((size_t)B * NB + A) * q + yy] = ((uint32_t)val[0][yy] << 16) | bits;
    }
    store_cell<I16>(table_out, n, r, c, val[a][y]);
    if (r == 0 && c == n && !hdr->invalid) *score = val[a][y];
}

static int pt_fold_enqueue(rna4r_ctx *ctx, const uint8_t *seq_dev, const int64_t *offset_dev, int n, int32_t *score_dev,
                           int32_t *status_dev, void *table_out, int table_dtype, void *ws, cudaStream_t st)
{
    const int q = ctx->q;
    PtWs w = pt_layout(ws, n, q);
    const int NB = n / q + 1;
    int launches = 0;
    RNA4R_CUDA(ctx, cudaMemsetAsync(w.hdr, 0, 256, st));
    encode_kernel<<<(NB * q + 1 + 255) / 256, 256, 0, st>>>(seq_dev, offset_dev, n, NB * q + 1, w.codes, w.hdr); ++launches;
    if (ctx->timing) RNA4R_CUDA(ctx, cudaEventRecord(ctx->ev0, st));
    for (int D = 0; D < NB; ++D) {
        if (table_dtype == RNA4R_TABLE_INT16)
            pt_tile_kernel<true><<<NB - D, q * q, 0, st>>>(n, q, D, NB, w.codes, ctx->R, w.H, w.V, w.hdr, score_dev, table_out);
        else
            pt_tile_kernel<false><<<NB - D, q * q, 0, st>>>(n, q, D, NB, w.codes, ctx->R, w.H, w.V, w.hdr, score_dev, table_out);
        ++launches;
    }
    if (ctx->timing) { RNA4R_CUDA(ctx, cudaEventRecord(ctx->ev1, st)); ctx->timing_valid = 1; }
    finish_kernel<<<1, 1, 0, st>>>(w.hdr, score_dev, status_dev, n); ++launches;
    RNA4R_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = launches;
    return RNA4R_OK;
}

// ====================================================================================================================
// RNA4R_ENGINE_MAXPLUS
// ====================================================================================================================
constexpr int MT = 32;      // tile side

struct MpWs {
    Hdr *hdr;
    int8_t *codes;      // [NT*32 + 1]
    int16_t *M;         // [NT*32][NT*32] row-major values, 0 where c <= r+1
    size_t bytes;
};
static inline MpWs mp_layout(void *base, int n)
{
    MpWs w;
    char *p = (char *)base;
    const size_t P = ((size_t)n / MT + 1) * MT;
    size_t off = 0;
    w.hdr = (Hdr *)(p + off); off += 256;
    w.codes = (int8_t *)(p + off); off += align_up(P + 16, 256);
    w.M = (int16_t *)(p + off); off += align_up(P * P * 2, 256);
    w.bytes = off;
    return w;
}

// one block (256 threads) <-> tile (I, I+D).  Bulk: C = max over the middle tiles K of M(I,K) (x) M(K,J) in max-plus,
// a thread owns 2 rows x 2 adjacent columns (one s16x2 pair per row).  Then the tile's own 63 anti-diagonals.
template <bool I16>
__global__ void __launch_bounds__(256) mp_tile_kernel(int n, int D, int P, const int8_t *__restrict__ codes, int16_t *__restrict__ M,
                                                      const Hdr *hdr, int32_t *score, void *table_out)
{
    __shared__ __align__(16) int16_t At[MT][MT + 2], Bt[MT][MT + 2];
    __shared__ int val[MT][MT + 1];
    const int tid = threadIdx.x;
    const int I = blockIdx.x, J = I + D;
    const int ty = tid / 16, tx = tid % 16;
    uint32_t acc0 = 0, acc1 = 0;                                   // rows 2ty, 2ty+1; columns 2tx | 2tx+1 << 16
    for (int K = I + 1; K <= J - 1; ++K) {
        for (int e = tid; e < MT * MT; e += 256) {
            const int rr = e / MT, cc = e % MT;
            At[rr][cc] = M[(size_t)(I * MT + rr) * P + K * MT + cc];
            Bt[rr][cc] = M[(size_t)(K * MT + rr) * P + J * MT + cc];
        }
        __syncthreads();
#pragma unroll 8
        for (int k = 0; k < MT; ++k) {
            const uint32_t b = *reinterpret_cast<const uint32_t *>(&Bt[k][2 * tx]);
            const uint32_t a0 = __byte_perm((uint32_t)(uint16_t)At[2 * ty][k], 0, 0x1010);
            const uint32_t a1 = __byte_perm((uint32_t)(uint16_t)At[2 * ty + 1][k], 0, 0x1010);
            acc0 = __viaddmax_s16x2(a0, b, acc0);                  // max(M(r,t) + M(t,c), acc) on two columns
            acc1 = __viaddmax_s16x2(a1, b, acc1);
        }
        __syncthreads();
    }
    val[2 * ty][2 * tx] = (int)(acc0 & 0xffffu); val[2 * ty][2 * tx + 1] = (int)(acc0 >> 16);
    val[2 * ty + 1][2 * tx] = (int)(acc1 & 0xffffu); val[2 * ty + 1][2 * tx + 1] = (int)(acc1 >> 16);
    if (D > 0) {
        for (int e = tid; e < MT * MT; e += 256) {
            const int rr = e / MT, cc = e % MT;
            At[rr][cc] = M[(size_t)(I * MT + rr) * P + I * MT + cc];      // diagonal tile (I,I): M(r,t), t in block I
            Bt[rr][cc] = M[(size_t)(J * MT + rr) * P + J * MT + cc];      // diagonal tile (J,J): M(t,c), t in block J
        }
    }
    __syncthreads();
    // closure: cell (a,y) on anti-diagonal s = (31-a) + y; one thread per cell of the anti-diagonal
    for (int s = 0; s <= 2 * MT - 2; ++s) {
        const int y = tid, a = MT - 1 - s + y;
        if (tid < MT && a >= 0 && a < MT) {
            const int r = I * MT + a, c = J * MT + y;
            int v;
            if (D == 0) {
                v = 0;
                if (y > a + 1) {
                    v = val[a + 1][y - 1] + rna4r_pair(codes[r], codes[c - 1]);
                    for (int t = a + 1; t < y; ++t) v = max(v, val[a][t] + val[t][y]);
                }
            } else {
                const int dl = (a < MT - 1 && y > 0) ? val[a + 1][y - 1] : (int)M[(size_t)(r + 1) * P + c - 1];
                v = max(val[a][y], dl + rna4r_pair(codes[r], codes[c - 1]));
                for (int t = a + 1; t < MT; ++t) v = max(v, (int)At[a][t] + val[t][y]);
                for (int t = 0; t < y; ++t) v = max(v, val[a][t] + (int)Bt[t][y]);
            }
            val[a][y] = v;
        }
        __syncthreads();
    }
    for (int e = tid; e < MT * MT; e += 256) {
        const int a = e / MT, y = e % MT;
        const int r = I * MT + a, c = J * MT + y;
        M[(size_t)r * P + c] = (int16_t)val[a][y];
        store_cell<I16>(table_out, n, r, c, val[a][y]);
        if (r == 0 && c == n && !hdr->invalid) *score = val[a][y];
    }
}

static int mp_fold_enqueue(rna4r_ctx *ctx, const uint8_t *seq_dev, const int64_t *offset_dev, int n, int32_t *score_dev,
                           int32_t *status_dev, void *table_out, int table_dtype, void *ws, cudaStream_t st)
{
    MpWs w = mp_layout(ws, n);
    const int NT = n / MT + 1, P = NT * MT;
    int launches = 0;
    RNA4R_CUDA(ctx, cudaMemsetAsync(ws, 0, w.bytes, st));          // header, and M = 0 on and below the diagonal band
    encode_kernel<<<(P + 1 + 255) / 256, 256, 0, st>>>(seq_dev, offset_dev, n, P + 1, w.codes, w.hdr); ++launches;
    if (ctx->timing) RNA4R_CUDA(ctx, cudaEventRecord(ctx->ev0, st));
    for (int D = 0; D < NT; ++D) {
        if (table_dtype == RNA4R_TABLE_INT16)
            mp_tile_kernel<true><<<NT - D, 256, 0, st>>>(n, D, P, w.codes, w.M, w.hdr, score_dev, table_out);
        else
            mp_tile_kernel<false><<<NT - D, 256, 0, st>>>(n, D, P, w.codes, w.M, w.hdr, score_dev, table_out);
        ++launches;
    }
    if (ctx->timing) { RNA4R_CUDA(ctx, cudaEventRecord(ctx->ev1, st)); ctx->timing_valid = 1; }
    finish_kernel<<<1, 1, 0, st>>>(w.hdr, score_dev, status_dev, n); ++launches;
    RNA4R_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = launches;
    return RNA4R_OK;
}

}  // namespace cmpeng
