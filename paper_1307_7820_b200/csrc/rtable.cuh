// rtable.cuh -- preprocessing kernels (step a2): the table R of PAPER.md:91-113.
#pragma once
#include "common.cuh"

// One thread per (v, vbar) pair runs the q-step black box of PAPER.md:94-111 ("embarrassingly
// parallel").  Index bit k of v / vbar is |v_k| / |vbar_k|.
// Consecutive threads take consecutive vbar, so the byte stores of a warp coalesce.
__global__ void rna4r_build_rtable_kernel(int q, uint8_t *__restrict__ R)
{
    const uint32_t N = 1u << q;
    const size_t total = (size_t)N * N;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const uint32_t v = (uint32_t)(e >> q), w = (uint32_t)(e & (N - 1));
        int maxval = 0, sum1 = 0, sum2 = 0;                 // line 1-2
        for (int k = 0; k < q; ++k) {                       // line 3
            sum1 += (int)((v >> k) & 1u);                   // line 4: v_k in {0,1}
            sum2 -= (int)((w >> k) & 1u);                   // line 5: vbar_k in {0,-1}
            if (sum1 + sum2 > maxval) maxval = sum1 + sum2; // line 6-7 (max-index: traceback, out of scope)
        }
        R[e] = (uint8_t)maxval;
    }
}

// Reachable quadrant: v_0 = vbar_0 = 0 by definition, so the fill only ever indexes
// even v and even vbar.  Rc[h][w] = R[2h][2w], h,w in [0, 2^(q-1)).  This 2^(2(q-1))-byte table is
// what the tiled engine keeps in shared memory (16 KB at q = 8: one row is 128 B = 32 banks).
__global__ void rna4r_build_compact_kernel(int q, const uint8_t *__restrict__ R, uint8_t *__restrict__ Rc)
{
    const int hb = q - 1;
    const uint32_t M = 1u << hb;
    const size_t total = (size_t)M * M;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const uint32_t h = (uint32_t)(e >> hb), w = (uint32_t)(e & (M - 1));
        Rc[e] = R[((size_t)(2 * h) << q) + 2 * w];
    }
}

// Ternary form of the same table for q >= 10, where 2^(2(q-1)) bytes no longer fit shared memory.  The listing
// PAPER.md:94-111 adds v_k and vbar_k in every step, so its result depends on the two vectors only through
// d_k = v_k - |vbar_k| in {-1, 0, 1}:  Rt[sum_{k=1}^{q-1} (d_k + 1) 3^(k-1)] = max(0, max_k sum_{k'<=k} d_k'),
// 3^(q-1) entries (19 683 at q = 10).  Entry (h, w) of Rc is Rt[sum_k (h_k + 1 - w_k) 3^(k-1)].
__global__ void rna4r_build_ternary_kernel(int q, uint32_t entries, uint8_t *__restrict__ Rt)
{
    for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < entries; e += gridDim.x * blockDim.x) {
        uint32_t x = e;
        int maxval = 0, sum = 0;                            // line 1-2; k = 0 adds v_0 + vbar_0 = 0
        for (int k = 1; k < q; ++k) {                       // line 3
            sum += (int)(x % 3u) - 1;                       // line 4-5: v_k + vbar_k
            x /= 3u;
            if (sum > maxval) maxval = sum;                 // line 6-7
        }
        Rt[e] = (uint8_t)maxval;
    }
}
