// common.cuh -- context, error handling and small device helpers shared by the rna4r kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/rna4r.h"

struct rna4r_ctx {
    uint32_t magic;
    int q;
    int device;
    int engine;              // resolved engine (never AUTO)
    int sm_count;
    uint8_t *R;              // device uint8[2^q][2^q]
    uint8_t *Rc;             // device uint8[2^(q-1)][2^(q-1)]   reachable quadrant, Rc[h][w] = R[2h][2w]
    uint8_t *Rt;             // device ternary-indexed table, 3^(q-1) entries (rtable.cuh), q = 9..11 only (else NULL)
    int last_launches;
    int last_cuda_error;
    int tiled_blocks_per_sm; // occupancy of the tiled fill kernel for this q (0 = not queried yet)
    int max_blocks_per_sm;   // rna4r_set_max_blocks_per_sm: cap on resident CTAs per SM of the fill kernel (0 = none)
    int max_blocks;          // rna4r_set_max_blocks: cap on the whole grid of the fill kernel (0 = none)
    int timing;              // record events around the dominant kernel
    int timing_valid;
    cudaEvent_t ev0, ev1;
    unsigned long long *trace;   // optional per-super-tile phase stamps (rna4r_set_trace)
    int trace_tiles;
    int engine_auto;         // the engine was left on (or set back to) RNA4R_ENGINE_AUTO: batches of short sequences take the SMEM engine
    int32_t *order_host;     // host scratch of the SMEM engine: sequence indices sorted by length (grown on demand)
    int order_cap;
    int32_t *route_host;     // host scratch of a batch split between the SMEM and the tiled engine: indices | lengths of the long part
    int route_cap;
};
// u64 words per super-tile in the optional trace buffer (rna4r_set_trace); a build with
// -DRNA4R_TRACE_WORDS=256 adds per-q-tile event stamps for tuning
#ifndef RNA4R_TRACE_WORDS
#define RNA4R_TRACE_WORDS 8
#endif
static const uint32_t RNA4R_MAGIC = 0x52344e41u;

// Checked build (-DRNA4R_CHECKS; tests and profiles/r02_sanitizer.md): every freshly computed cell must differ from its
// finished neighbours by 0 or 1 (Lemma 1), packed offsets must fit their fields and table indices the
// table.  A cell computed from operands that another warp / CTA had not finished yet breaks Lemma 1 with high
// probability, so this traps on ordering bugs of the flag / barrier protocols as well as on out-of-range indices.
#ifdef RNA4R_CHECKS
#define RNA4R_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define RNA4R_CHECK(cond) do { } while (0)
#endif

#define RNA4R_CUDA(ctx, call)                                             \
    do {                                                                  \
        cudaError_t e__ = (call);                                         \
        if (e__ != cudaSuccess) {                                         \
            if (ctx) (ctx)->last_cuda_error = (int)e__;                   \
            return RNA4R_ERR_CUDA;                                        \
        }                                                                 \
    } while (0)

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// base byte -> code 0..3 (A,C,G,U/T, either case); 4 = not a base (reading g4)
__device__ __forceinline__ int rna4r_base_code(uint8_t c)
{
    switch (c) {
    case 'A': case 'a': return 0;
    case 'C': case 'c': return 1;
    case 'G': case 'g': return 2;
    case 'U': case 'u': case 'T': case 't': return 3;
    default: return 4;
    }
}
// b(x,y) of eq. (1): A-U and C-G pair; code 4 (padding / invalid) pairs with nothing
__device__ __forceinline__ int rna4r_pair(int x, int y) { return (x + y == 3) ? 1 : 0; }

__device__ __forceinline__ unsigned long long global_timer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ int ld_acquire_gpu(const int *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu(int *p, int v)
{
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
