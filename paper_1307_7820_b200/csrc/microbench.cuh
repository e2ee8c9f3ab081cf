// microbench.cuh -- measured ceilings of the lookup sequence (a profiling aid: "measure INT issue rate
// with a microbenchmark on the box rather than assuming it").
//
// The roofline of this path is quoted against the shared-memory formula  #SMs x 32 lanes x f_SM  lookups/s (one
// 32-lane gather wavefront per SM per clock).  One lookup is, however, FOUR warp instructions (add W+X, LEA.HI for the
// address, LDS.U8, VIADDMNMX.U16x2 -- tiled_engine.cuh lookup_max) on an SM that issues four warp instructions per
// clock, so the issue slots bind at the same rate as the shared-memory pipe and every operand load or loop instruction
// comes off the top.  These kernels run exactly that sequence from every SM, conflict-free, and report what the
// hardware sustains:
//   variant 0  "pure":    operands in registers, 16 independent lookups per loop trip (the instruction floor);
//   variant 1  "product": tiled::product_accumulate as the bulk product runs it (row words by broadcast LDS.128,
//                         column words per lane, 16 lookups per 2 + 2 operand loads) on a resident panel pair;
//   variant 2  "ternary": variant 0 on the q = 10 table of 3^9 entries (same four instructions), operands in registers.
#pragma once
#include "tiled_engine.cuh"

namespace microbench {

using tiled::Cfg;
using tiled::Smem;

// Stage the table exactly as fill_kernel does (same pitch), from the context's compact table.
template <int Q>
__device__ __forceinline__ void stage_table(const Smem<Q> &sm, const uint8_t *tbl, int tid, int nthr)
{
    using C = Cfg<Q>;
    constexpr int ROWB = 1 << C::HB;
    if constexpr (C::TERN) {
        const uint4 *src = reinterpret_cast<const uint4 *>(tbl);
        uint4 *dst = reinterpret_cast<uint4 *>(sm.tbl);
        for (int e = tid; e < (C::TBL_BYTES + 15) / 16; e += nthr) dst[e] = __ldg(src + e);
    } else {
        for (int e = tid; e < ROWB * ROWB; e += nthr) sm.tbl[(e / ROWB) * C::TBL_PITCH + e % ROWB] = tbl[e];
    }
}

template <int Q, int VARIANT>
__global__ void __launch_bounds__(256) lookup_kernel(const uint8_t *__restrict__ tbl, int iters, uint32_t *__restrict__ sink)
{
    using C = Cfg<Q>;
    extern __shared__ __align__(16) uint8_t smem_raw[];
    Smem<Q> sm(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    stage_table<Q>(sm, tbl, tid, blockDim.x);
    // operand panels for variant 1: row words share h per row (warp-uniform loads), column words spread v over the lanes
    for (int e = tid; e < 2 * C::PANEL_WORDS; e += blockDim.x) {
        const bool is_col = e >= C::PANEL_WORDS;
        const uint32_t k = (uint32_t)(e % C::T), g = (uint32_t)((e % C::PANEL_WORDS) / C::T);
        const uint32_t bits = (k * 5u + g * 3u) & ((1u << C::HB) - 1u);
        sm.stg[e] = is_col ? ((bits << C::ISHIFT) | ((k + g) << C::VSHIFT))
                           : (((bits * (uint32_t)C::TBL_PITCH) << C::ISHIFT) | ((2u * k + g) << C::VSHIFT));
    }
    __syncthreads();
    uint32_t total = 0;
    if constexpr (VARIANT == 1) {
        uint32_t acc[2][C::RPT];
#pragma unroll
        for (int rr = 0; rr < C::RPT; ++rr) acc[0][rr] = acc[1][rr] = 0;
        const int t = tid % C::PTHR;
        const int cj = t % C::HT, rb = t / C::HT;
        for (int it = 0; it < iters; ++it) tiled::product_accumulate<Q>(sm, 0, acc, cj, rb);      // 8 groups x 2 x RPT lookups
#pragma unroll
        for (int rr = 0; rr < C::RPT; ++rr) total += acc[0][rr] + acc[1][rr];
    } else {
        // 16 row words per warp (distinct h, same for every lane), one column word per lane (distinct v: distinct banks)
        uint32_t w[16], acc[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const uint32_t h = (uint32_t)(warp * 16 + k) & ((1u << C::HB) - 1u);
            w[k] = ((h * (uint32_t)C::TBL_PITCH) << C::ISHIFT) | ((uint32_t)k << C::VSHIFT);
            acc[k] = 0;
        }
        uint32_t x = ((uint32_t)(lane * 4 + (warp & 3)) & ((1u << C::HB) - 1u)) << C::ISHIFT;
        const uint32_t dx = 1u << C::VSHIFT;             // the value field moves, the gather address does not
        for (int it = 0; it < iters; ++it) {
            x += dx;
#pragma unroll
            for (int k = 0; k < 16; ++k) acc[k] = tiled::lookup_max<Q>(sm, w[k] + x, acc[k]);
        }
#pragma unroll
        for (int k = 0; k < 16; ++k) total += acc[k];
    }
    if (total == 0x7fffffffu) sink[0] = total;           // keeps the loop alive; never true for these operands
}

template <int Q, int VARIANT>
static int run(rna4r_ctx *ctx, int iters, int blocks_per_sm, uint32_t *sink, cudaStream_t st, float *ms, double *lookups)
{
    using C = Cfg<Q>;
    RNA4R_CUDA(ctx, cudaFuncSetAttribute(lookup_kernel<Q, VARIANT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES));
    int fit = 0;
    RNA4R_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&fit, lookup_kernel<Q, VARIANT>, 256, C::SMEM_BYTES));
    if (fit < 1) return RNA4R_ERR_CUDA;
    if (blocks_per_sm < 1 || blocks_per_sm > fit) blocks_per_sm = fit;
    const int blocks = ctx->sm_count * blocks_per_sm;
    cudaEvent_t e0, e1;
    RNA4R_CUDA(ctx, cudaEventCreate(&e0));
    RNA4R_CUDA(ctx, cudaEventCreate(&e1));
    const uint8_t *tbl = C::TERN ? ctx->Rt : ctx->Rc;
    lookup_kernel<Q, VARIANT><<<blocks, 256, C::SMEM_BYTES, st>>>(tbl, iters / 8 + 1, sink);     // warm-up
    cudaEventRecord(e0, st);
    lookup_kernel<Q, VARIANT><<<blocks, 256, C::SMEM_BYTES, st>>>(tbl, iters, sink);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return RNA4R_ERR_CUDA; }
    const double per_thread = (VARIANT == 1) ? 8.0 * 2.0 * C::RPT : 16.0;
    *lookups = (double)blocks * 256.0 * per_thread * (double)iters;
    return RNA4R_OK;
}

}  // namespace microbench
