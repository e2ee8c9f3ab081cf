// diag_engine.cuh -- RNA4R_ENGINE_DIAG: the parallel two-vector algorithm exactly as section 4 of
// the paper states it: one "process" (thread) per cell of the current
// anti-diagonal, one launch (= one synchronisation) per diagonal, floor((j-i)/q)
// lookups with groups aligned relative to i (reading g19) then a < q residual loop, and per-cell
// sliding difference vectors d_H, d_V updated in O(1) by shift-and-append.
// It is the paper-literal comparison point and the engine for q = 11, 12; the B200 design is
// tiled_engine.cuh.
//
// The only liberty taken is the storage layout: all three per-cell arrays (D, d_H, d_V) are
// stored DIAGONAL-MAJOR, element (row r, column c) at [c - r + 1][r], pitch n + 2.  Then for a
// fixed group k' the threads i = 1, 2, ... of a warp read consecutive addresses both for the row
// operand (i, i + k'q) and for the column operand (i + k'q + 1, i + d): every stream coalesces.
#pragma once
#include "common.cuh"

struct DiagWs {
    int8_t *codes;     // [n + 2], 1-based
    int *invalid;      // [1]
    uint16_t *hrun;    // [n + 2] running horizontal window of row i
    uint16_t *vrun;    // [n + 2] running vertical window of column j
    int16_t *Dd;       // [(n + 1) * (n + 2)] diagonal-major D
    uint16_t *Hd;      // d_H(i,c): vector of cells D(i, c..c+q-1), diagonal-major at (i, c)
    uint16_t *Vd;      // d_V(i,j): vector of cells D(i..i+q-1, j), diagonal-major at (i, j)
    size_t bytes;
};

static inline DiagWs diag_ws_layout(void *base, int n)
{
    DiagWs w;
    char *p = (char *)base;
    size_t off = 0;
    const size_t P = (size_t)n + 2;
    w.invalid = (int *)(p + off); off += 256;
    w.hrun = (uint16_t *)(p + off); off += align_up(P * 2, 256);
    w.vrun = (uint16_t *)(p + off); off += align_up(P * 2, 256);
    w.codes = (int8_t *)(p + off); off += align_up(P, 256);
    w.Dd = (int16_t *)(p + off); off += align_up((size_t)(n + 1) * P * 2, 256);
    w.Hd = (uint16_t *)(p + off); off += align_up((size_t)(n + 1) * P * 2, 256);
    w.Vd = (uint16_t *)(p + off); off += align_up((size_t)(n + 1) * P * 2, 256);
    w.bytes = off;
    return w;
}

// `offset` (device, may be NULL): offset[0] = start of the sequence in seq, offset[1] = its end (a batch member);
// a length that disagrees with n (from lens_host) is reported instead of read (RNA4R_STATUS_BAD_OFFSETS).
__global__ void diag_encode_kernel(const uint8_t *__restrict__ seq, const int64_t *__restrict__ offset, int n,
                                   int8_t *__restrict__ codes, int *invalid)
{
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    int64_t start = 0;
    if (offset) {
        start = offset[0];
        if (offset[1] - start != (int64_t)n) { if (t == 0) atomicOr(invalid, RNA4R_STATUS_BAD_OFFSETS); codes[t + 1] = 4; return; }
    }
    int c = rna4r_base_code(seq[start + t]);
    if (c == 4) atomicOr(invalid, RNA4R_STATUS_BAD_BASE);
    codes[t + 1] = (int8_t)c;
}

// One anti-diagonal d = j - i (1 <= d <= n-1); thread <-> cell (i, i+d), i = 1..n-d.
__global__ void diag_fill_kernel(int n, int q, int d, const int8_t *__restrict__ codes,
                                 const uint8_t *__restrict__ R,
                                 int16_t *__restrict__ Dd, uint16_t *__restrict__ Hd, uint16_t *__restrict__ Vd,
                                 uint16_t *__restrict__ hrun, uint16_t *__restrict__ vrun)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x + 1;
    if (i > n - d) return;
    const int j = i + d;
    const size_t P = (size_t)n + 2;
#define AT(dd, r) ((size_t)((dd) + 1) * P + (size_t)(r))
    // PAPER.md:234  D(i,j) <- D(i+1,j-1) + b(S[i],S[j])
    int best = (int)Dd[AT(d - 2, i + 1)] + rna4r_pair(codes[i], codes[j]);
    // PAPER.md:254-260  k' = 0 .. floor((j-i)/q)-1, k = i + k'q:
    //   D(i,j) = max{D(i,j), D(i,k) + D(k+1,j) + R[d_H(i,k)][d_V(k+1,j)]}
    const int ngroups = d / q;
    for (int kp = 0; kp < ngroups; ++kp) {
        const int off = kp * q;                       // k = i + off
        const int a = Dd[AT(off, i)];                 // D(i,k)
        const int b = Dd[AT(d - off - 1, i + off + 1)];   // D(k+1,j)
        const uint32_t hv = Hd[AT(off, i)];           // d_H(i,k)
        const uint32_t vv = Vd[AT(d - off - 1, i + off + 1)];   // d_V(k+1,j)
        const int c = a + b + (int)__ldg(R + ((size_t)hv << q) + vv);
        best = max(best, c);
    }
    // PAPER.md:261-263  residual k = i + floor((j-i)/q) q .. j-1
    for (int off = ngroups * q; off < d; ++off) {
        const int c = (int)Dd[AT(off, i)] + (int)Dd[AT(d - off - 1, i + off + 1)];
        best = max(best, c);
    }
    Dd[AT(d, i)] = (int16_t)best;
    // PAPER.md:264-267  shift the previous difference vector and append the new difference.
    const uint32_t mask = (1u << q) - 1u;
    const uint32_t hbit = (uint32_t)(best - (int)Dd[AT(d - 1, i)]);        // D(i,j) - D(i,j-1)
    const uint32_t vbit = (uint32_t)(best - (int)Dd[AT(d - 1, i + 1)]);    // D(i,j) - D(i+1,j)
    // horizontal window ending at j: bit p = D(i,j-q+1+p) - D(i,j-q+p), p = 1..q-1, bit 0 = v_0 = 0
    const uint32_t h = (((uint32_t)hrun[i] >> 1) | (hbit << (q - 1))) & mask & ~1u;
    hrun[i] = (uint16_t)h;
    if (d - q + 1 >= 0) Hd[AT(d - q + 1, i)] = (uint16_t)h;                 // d_H(i, j-q+1)
    // vertical window starting at i: bit p = D(i+p-1,j) - D(i+p,j), p = 1..q-1, bit 0 = vbar_0 = 0
    const uint32_t v = (((uint32_t)vrun[j] << 1) | (vbit << 1)) & mask & ~1u;
    vrun[j] = (uint16_t)v;
    Vd[AT(d, i)] = (uint16_t)v;                                             // d_V(i, j)
#undef AT
}

// D(1,n) -> score (or -1), and the optional row-major table.
__global__ void diag_score_kernel(int n, const int16_t *__restrict__ Dd, const int *invalid, int32_t *score, int32_t *status)
{
    const size_t P = (size_t)n + 2;
    *score = *invalid ? -1 : (int32_t)Dd[(size_t)n * P + 1];   // diagonal n-1, row 1
    if (status) *status = *invalid;
}
__global__ void diag_empty_kernel(const int64_t *__restrict__ offset, int32_t *score, int32_t *status)
{
    const int bad = (offset && offset[1] != offset[0]) ? RNA4R_STATUS_BAD_OFFSETS : 0;
    *score = bad ? -1 : 0;
    if (status) *status = bad;
}

template <typename OutT>
__global__ void diag_table_kernel(int n, const int16_t *__restrict__ Dd, OutT *__restrict__ out)
{
    const size_t P = (size_t)n + 2;
    const size_t total = (size_t)n * n;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const int r = (int)(e / n) + 1, c = (int)(e % n) + 1;
        out[e] = (c >= r) ? (OutT)Dd[(size_t)(c - r + 1) * P + r] : (OutT)0;
    }
}

static int diag_fold_enqueue(rna4r_ctx *ctx, const uint8_t *seq_dev, const int64_t *offset_dev, int n, int32_t *score_dev,
                             int32_t *status_dev, void *table_out, int table_dtype, void *ws, cudaStream_t st)
{
    DiagWs w = diag_ws_layout(ws, n);
    const size_t P = (size_t)n + 2;
    int launches = 0;
    // zero: invalid flag, hrun, vrun, codes, and the two zero diagonals D(i,i-1) = D(i,i) = 0
    RNA4R_CUDA(ctx, cudaMemsetAsync(ws, 0, (size_t)((char *)w.Dd - (char *)ws) + 2 * P * sizeof(int16_t), st));
    if (n > 0) {
        diag_encode_kernel<<<(n + 255) / 256, 256, 0, st>>>(seq_dev, offset_dev, n, w.codes, w.invalid);
        ++launches;
    }
    const int q = ctx->q;
    if (ctx->timing) RNA4R_CUDA(ctx, cudaEventRecord(ctx->ev0, st));
    for (int d = 1; d <= n - 1; ++d) {
        const int cells = n - d;
        diag_fill_kernel<<<(cells + 127) / 128, 128, 0, st>>>(n, q, d, w.codes, ctx->R, w.Dd, w.Hd, w.Vd, w.hrun, w.vrun);
        ++launches;
    }
    if (ctx->timing) { RNA4R_CUDA(ctx, cudaEventRecord(ctx->ev1, st)); ctx->timing_valid = 1; }
    if (n == 0) {
        diag_empty_kernel<<<1, 1, 0, st>>>(offset_dev, score_dev, status_dev);
        ++launches;
    } else {
        diag_score_kernel<<<1, 1, 0, st>>>(n, w.Dd, w.invalid, score_dev, status_dev);
        ++launches;
    }
    if (table_out && n > 0) {
        const int blocks = (int)(((size_t)n * n + 255) / 256 > 65535 * 4 ? 65535 * 4 : ((size_t)n * n + 255) / 256);
        if (table_dtype == RNA4R_TABLE_INT16)
            diag_table_kernel<int16_t><<<blocks, 256, 0, st>>>(n, w.Dd, (int16_t *)table_out);
        else
            diag_table_kernel<int32_t><<<blocks, 256, 0, st>>>(n, w.Dd, (int32_t *)table_out);
        ++launches;
    }
    RNA4R_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = launches;
    return RNA4R_OK;
}
