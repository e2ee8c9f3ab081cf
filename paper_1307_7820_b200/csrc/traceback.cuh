// traceback.cuh -- one optimal structure from a finished table.
//
// The paper keeps arg-max indices beside the maxima (D*).  Here the pairs are recovered by
// re-running eq. (1) along the optimal path of the stored table D, which needs no second
// table:  an interval (i,j) with D(i,j) > 0 either
//   pairs its ends      -- b(S_i,S_j) = 1 and D(i,j) = 1 + D(i+1,j-1): record (i,j), continue with (i+1,j-1);
//   or splits           -- the smallest k in [i+1, j] with D(i,j) = D(i,k-1) + D(k,j): continue with (k,j),
//                          hand (i,k-1) to the work queue.
// The intervals of one structure form a tree; its branches are independent, so the traceback is a parallel
// depth-first walk: every warp owns one interval at a time, follows the pair chain and the right child itself
// and publishes the left child in a ticket queue (head/tail counters, one slot per ticket, written once).
// `pending` counts intervals that are queued or being walked; 0 = done.  The k search reads D(i,k-1) along
// row i (coalesced) and D(k,j) along column j, 32 candidates per step, and stops at the first hit.
// The rule (pair first, then smallest k) makes the structure deterministic; any rule gives D(1,n) pairs.
#pragma once
#include "common.cuh"

namespace traceback {

struct Queue {
    int head;       // next ticket to pop
    int tail;       // next ticket to push
    int pending;    // intervals queued or being walked
    int npairs;
    int invalid;    // the sequence holds a byte that is not a base
    int pad[3];
};

static inline size_t workspace_bytes(int n) { return 256 + ((size_t)2 * (size_t)n + 64) * sizeof(unsigned long long); }

template <typename TT>
__device__ __forceinline__ int getD(const TT *tab, int n, int i, int j)      // 1-based, D(i,j) = 0 for j <= i
{
    return (j <= i) ? 0 : (int)tab[(size_t)(i - 1) * n + (j - 1)];
}

constexpr unsigned long long EMPTY = ~0ull;

__global__ void init_kernel(Queue *q, unsigned long long *slots, int nslots, int32_t *pairs, int n)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    for (int e = t; e < nslots; e += gridDim.x * blockDim.x) slots[e] = EMPTY;
    for (int e = t; e < n; e += gridDim.x * blockDim.x) pairs[e] = -1;
    if (t == 0) {
        q->head = 0; q->npairs = 0; q->invalid = 0;
        if (n >= 2) { slots[0] = ((unsigned long long)1 << 32) | (unsigned)n; q->tail = 1; q->pending = 1; }
        else { q->tail = 0; q->pending = 0; }
    }
}

template <typename TT>
__global__ void __launch_bounds__(256) walk_kernel(const uint8_t *seq, int n, const TT *tab, Queue *q,
                                                   unsigned long long *slots, int32_t *pairs)
{
    const int lane = threadIdx.x & 31;
    constexpr unsigned FULL = 0xffffffffu;
    for (;;) {
        // ---- pop one interval (lane 0 takes a ticket and waits for its slot, or for the end)
        unsigned long long item = EMPTY;
        if (lane == 0) {
            int ticket = -1;
            for (;;) {
                if (*(volatile int *)&q->pending <= 0) break;
                if (ticket < 0) {
                    const int h = *(volatile int *)&q->head;
                    if (h < *(volatile int *)&q->tail) { if (atomicCAS(&q->head, h, h + 1) == h) ticket = h; }
                    else __nanosleep(200);
                    continue;
                }
                item = *(volatile unsigned long long *)&slots[ticket];
                if (item != EMPTY) break;
                __nanosleep(100);
            }
        }
        item = __shfl_sync(FULL, item, 0);
        if (item == EMPTY) return;
        int i = (int)(item >> 32), j = (int)(item & 0xffffffffu);
        int found = 0;
        // ---- walk: pair chain and right children here, left children to the queue
        while (j > i) {
            const int v = getD(tab, n, i, j);
            if (v == 0) break;
            const int ci = rna4r_base_code(seq[i - 1]), cj = rna4r_base_code(seq[j - 1]);
            if ((ci == 4 || cj == 4) && lane == 0) q->invalid = 1;
            if (rna4r_pair(ci, cj) && v == 1 + getD(tab, n, i + 1, j - 1)) {
                if (lane == 0) { pairs[i - 1] = j - 1; pairs[j - 1] = i - 1; }
                ++found; ++i; --j;
                continue;
            }
            int k = -1;
            for (int k0 = i + 1; k0 <= j && k < 0; k0 += 32) {
                const int kk = k0 + lane;
                const bool hit = kk <= j && getD(tab, n, i, kk - 1) + getD(tab, n, kk, j) == v;
                const unsigned m = __ballot_sync(FULL, hit);
                if (m) k = k0 + __ffs(m) - 1;
            }
            if (k < 0) { if (lane == 0) q->invalid = 2; break; }       // not a table of eq. (1)
            // left child (i, k-1) -> queue if it can hold a pair; right child (k, j) continues here
            if (k - 1 > i && getD(tab, n, i, k - 1) > 0 && lane == 0) {
                atomicAdd(&q->pending, 1);
                const int t = atomicAdd(&q->tail, 1);
                *(volatile unsigned long long *)&slots[t] = ((unsigned long long)i << 32) | (unsigned)(k - 1);
                __threadfence();
            }
            i = k;
        }
        if (lane == 0) {
            if (found) atomicAdd(&q->npairs, found);
            __threadfence();
            atomicSub(&q->pending, 1);
        }
    }
}

__global__ void finish_kernel(const Queue *q, int32_t *npairs_out)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) *npairs_out = q->invalid ? -1 : q->npairs;
}

}  // namespace traceback
