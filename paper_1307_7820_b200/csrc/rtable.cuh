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

// Nibble packing of Rc for q where the byte table no longer fits shared memory (q = 10: 2^18
// entries, values 0..9 -> 128 KB).  Entry e lives in byte e/2, low nibble for even e.
__global__ void rna4r_pack_nibbles_kernel(size_t entries, const uint8_t *__restrict__ Rc, uint8_t *__restrict__ Rc4)
{
    for (size_t b = (size_t)blockIdx.x * blockDim.x + threadIdx.x; b < entries / 2; b += (size_t)gridDim.x * blockDim.x)
        Rc4[b] = (uint8_t)((Rc[2 * b] & 15) | ((Rc[2 * b + 1] & 15) << 4));
}
