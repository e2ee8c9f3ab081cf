/*
 * rna4r.h -- C ABI of the B200-native two-vector Four-Russians RNA fold.
 *
 * Source of every operation: Venkatachalam, Gusfield, Frid, "Faster Algorithms for RNA-folding
 * using the Four-Russians method" (arxiv 1307.7820), cited below as PAPER.md:<line>.
 *
 * Problem (section 2): input a sequence S[1..n] over {A,C,G,U}; output D(1,n),
 * the largest number of non-crossing complementary (A-U, C-G) base pairs, where
 *     D(i,i-1) = D(i,i) = 0,
 *     D(i,j)   = max{ b(S_i,S_j) + D(i+1,j-1),  max_{i+1<=k<=j} D(i,k-1) + D(k,j) }      (eq. (1))
 * and, on request, the whole upper-triangular table D.
 *
 * Method (PAPER.md:62-123 section 3.1, :221-269 section 4): by Lemma 1 adjacent
 * cells of a row / column differ by 0 or 1, so q consecutive cells are an anchor plus a q-bit
 * difference vector (v_0 = 0 by definition); eq. (3) replaces q
 * steps of the inner max by  D(i,l) + D(l+1,j) + R[v][vbar]  with R tabulated once for all
 * 2^q x 2^q vector pairs.  The fill runs as an anti-diagonal wavefront
 * (PAPER.md:223-245).
 *
 * General rules of this ABI
 *   - Every pointer argument says "host" or "device".  Device pointers are plain CUDA device
 *     addresses on the context's device; the caller allocates and owns ALL device buffers
 *     (sequence, outputs, workspace) and the stream.  The library allocates only what
 *     rna4r_prepare creates (the R tables) and frees it in rna4r_destroy.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - rna4r_fold / rna4r_fold_batch only ENQUEUE work on `stream` and return; they never allocate
 *     device memory and never synchronise.  (rna4r_fold_batch keeps two small context-owned HOST
 *     index arrays -- the batch sorted by length, the sequences routed to the tiled engine -- which
 *     grow when a batch holds more sequences than any before.)  The *_host variants copy in/out and
 *     synchronise `stream`.
 *   - A workspace size is valid for the engine setting it was asked with (rna4r_set_engine).
 *   - Every function returns 0 (RNA4R_OK) or a negative RNA4R_ERR_* code; nothing throws.
 *   - There is NO CPU fallback: on a machine without an sm_100 device rna4r_prepare fails with
 *     RNA4R_ERR_DEVICE and nothing else can be called.
 *   - Results are deterministic integers (max is order independent): same input, same bits.
 *   - Input alphabet: bytes A C G U, lower case accepted, T == U.  Any other byte makes that
 *     sequence's score -1 (and, for rna4r_fold, leaves table_out unspecified); other sequences
 *     of a batch are unaffected.  n = 0 and n = 1 are valid and score 0.
 *   - Errors that only the device can see (a byte that is not a base; device offsets that disagree
 *     with lens_host) never fail the call: the sequence's score is -1 and, when the caller passes a
 *     status array (rna4r_fold_batch_status), its status word holds the RNA4R_STATUS_* bits.  A
 *     single fold (rna4r_fold) reports through the score alone: -1 means RNA4R_STATUS_BAD_BASE.
 */
#ifndef RNA4R_H
#define RNA4R_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- error codes ---- */
#define RNA4R_OK              0
#define RNA4R_ERR_BAD_Q      -1   /* q outside 2..12                                           */
#define RNA4R_ERR_NULL       -2   /* a required pointer is NULL                                */
#define RNA4R_ERR_BAD_N      -3   /* n < 0, count < 0, or n too large for the chosen engine/q  */
#define RNA4R_ERR_WORKSPACE  -4   /* workspace_bytes smaller than rna4r_workspace_bytes(...)   */
#define RNA4R_ERR_CONTEXT    -5   /* NULL / destroyed context                                  */
#define RNA4R_ERR_CUDA       -6   /* a CUDA runtime call failed (see rna4r_last_cuda_error)    */
#define RNA4R_ERR_DEVICE     -7   /* no CUDA device, or the device is not compute capability 10.x */
#define RNA4R_ERR_DTYPE      -8   /* table_dtype not one of RNA4R_TABLE_*                      */
#define RNA4R_ERR_ENGINE     -9   /* engine id unknown, or the engine does not support this q  */
#define RNA4R_ERR_SETUP      -10  /* rna4r_fold_static before rna4r_fold_static_setup on this device */

/* ---- per-sequence status bits (device-detected; see rna4r_fold_batch_status) ---- */
#define RNA4R_STATUS_OK           0
#define RNA4R_STATUS_BAD_BASE     1   /* the sequence holds a byte outside A C G U T (either case)          */
#define RNA4R_STATUS_BAD_OFFSETS  2   /* offsets_dev[t+1]-offsets_dev[t] != lens_host[t]: sequence not read */

/* ---- rna4r_workspace_bytes flags ---- */
#define RNA4R_WS_DEVICE        0      /* device-buffer calls (rna4r_fold, rna4r_fold_batch)                 */
#define RNA4R_WS_HOST_STAGING  1      /* + staging for the *_host variants (bases, offsets, scores)        */
#define RNA4R_WS_HOST_TABLE16  2      /* + staging for rna4r_fold_host's int16 table (count == 1 only)     */
#define RNA4R_WS_HOST_TABLE32  4      /* + staging for rna4r_fold_host's int32 table (count == 1 only)     */

/* ---- table_out element types ---- */
#define RNA4R_TABLE_NONE   0
#define RNA4R_TABLE_INT16  1      /* exact for n <= 65534 (D <= n/2)  */
#define RNA4R_TABLE_INT32  2

/* ---- fill engines ---- */
#define RNA4R_ENGINE_AUTO   0     /* TILED when 2 <= q <= 11, else DIAG; for 4 <= q <= 8 rna4r_fold_batch folds
                                     the sequences of at most rna4r_smem_max_n(ctx) bases on SMEM and the
                                     longer ones of the same batch on TILED                             */
#define RNA4R_ENGINE_TILED  1     /* persistent super-tile wavefront, R resident in shared memory
                                     (the B200 design); q in 2..11 (q = 9..11
                                     index the table in base 3, see rna4r_table_to_host)        */
#define RNA4R_ENGINE_DIAG   2     /* paper-literal section 4 algorithm: one launch per anti-
                                     diagonal, one thread per cell, per-cell sliding vectors
                                     (PAPER.md:249-267); any q in 2..12; the comparison point   */

#define RNA4R_ENGINE_SMEM   3     /* one CTA per sequence, the whole fold's row / column words resident
                                     in shared memory (batches of short sequences, BASELINE.json
                                     configs[3]); q in 4..8, n <= rna4r_smem_max_n */

#define RNA4R_ENGINE_PAPER_TILE 4  /* the paper's own CUDA design, section 5.3: one block per
                                     q x q tile, one launch per tile-diagonal, only differences (+ anchors)
                                     stored, H vectors row-major by tile, V vectors column-major by tile, R in
                                     global memory; any q in 2..12; a comparison point                       */
#define RNA4R_ENGINE_MAXPLUS 5    /* no Four-Russians table: eq. (1) as a blocked max-plus
                                     closure on int16 values with DPX add-max, one launch per 32 x 32 tile-
                                     diagonal; q is ignored; a comparison point           */

typedef struct rna4r_ctx rna4r_ctx;   /* opaque; owns the device R tables for one q on one device */

/*
 * rna4r_prepare -- preprocessing step ("we will run the above algorithm for all
 * possible vector pairs of length q and store the results in table R"; the
 * 2^q x 2^q entries are independent).  Builds on `device`, enqueued on `stream`:
 *   - R : uint8[2^q][2^q], R[v][vbar] = max-val of the listing PAPER.md:94-111, index bit k = |v_k|;
 *   - the compact reachable quadrant the fill kernels stage in shared memory
 *     (v_0 = vbar_0 = 0): Rc[h][w] = R[2h][2w], 2^(q-1) x 2^(q-1) entries.
 * q: host int, 2..12.  device: CUDA ordinal.  out: host pointer receiving the context.
 * Errors: BAD_Q, NULL, DEVICE, CUDA.
 */
int rna4r_prepare(int q, int device, void *stream, rna4r_ctx **out);

/* Frees the context and its device tables (synchronises the device).  Errors: CONTEXT. */
int rna4r_destroy(rna4r_ctx *ctx);

/* q of the context (or RNA4R_ERR_CONTEXT). */
int rna4r_q(const rna4r_ctx *ctx);

/* Device pointer to R (uint8[2^q][2^q], row = horizontal vector v, column = vertical vector vbar),
 * or NULL.  Valid until rna4r_destroy; ordered after rna4r_prepare's stream work. */
const uint8_t *rna4r_table(const rna4r_ctx *ctx);

/* Device pointer to the compact table Rc (uint8[2^(q-1)][2^(q-1)]), or NULL. */
const uint8_t *rna4r_table_compact(const rna4r_ctx *ctx);

/* Copies R (compact = 0: 2^q * 2^q bytes), Rc (compact = 1: 2^(q-1) * 2^(q-1) bytes) or the ternary-indexed
 * form Rt (compact = 2: 3^(q-1) bytes; exists for q = 9, 10 and 11 only, otherwise RNA4R_ERR_ENGINE) into HOST
 * memory dst_host after synchronising the device (a test / inspection helper).  The black box
 * adds v_k and vbar_k in every step, so max-val depends on the pair only through d_k = v_k + vbar_k in
 * {-1, 0, 1}:  Rt[sum_{k=1}^{q-1} (d_k + 1) 3^(k-1)] = R[v][vbar] with bit k of v = v_k, bit k of vbar = |vbar_k|.
 * Errors: CONTEXT, NULL, BAD_N (compact not 0..2), ENGINE, CUDA. */
int rna4r_table_to_host(rna4r_ctx *ctx, uint8_t *dst_host, int compact);

/* Selects the fill engine (RNA4R_ENGINE_*) for later fold calls.  Errors: CONTEXT, ENGINE. */
int rna4r_set_engine(rna4r_ctx *ctx, int engine);
int rna4r_engine(const rna4r_ctx *ctx);   /* the engine fold calls will use (resolved, never AUTO) */
/* Longest sequence RNA4R_ENGINE_SMEM folds for the context's q (its state has to fit 227 KB of shared memory),
 * -1 if the engine does not support this q, or RNA4R_ERR_CONTEXT. */
int rna4r_smem_max_n(const rna4r_ctx *ctx);

/*
 * Workspace size in bytes for `count` sequences each of length <= n_max with the context's current
 * engine (an upper bound; 0 on error).  flags: RNA4R_WS_DEVICE, or RNA4R_WS_HOST_* bits OR-ed to add
 * the staging area of the *_host variants.  rna4r_workspace_bytes_batch gives the exact device-side
 * size for given lengths (lens_host: host int32[count]); rna4r_workspace_bytes_host (below) the exact
 * size for the *_host variants.  The workspace needs 256-byte alignment and holds only scratch: its
 * contents are undefined before and after a call.
 */
size_t rna4r_workspace_bytes(const rna4r_ctx *ctx, int n_max, int count, int flags);
size_t rna4r_workspace_bytes_batch(const rna4r_ctx *ctx, const int32_t *lens_host, int count);

/*
 * Caps the number of CTAs per SM the persistent fill kernel of the TILED engine is launched with
 * (a tuning / test knob: a smaller grid changes the interleaving of the wavefront tasks, never the
 * result).  0 = no cap (the default: as many as fit).  Errors: CONTEXT, BAD_N (negative).
 */
int rna4r_set_max_blocks_per_sm(rna4r_ctx *ctx, int blocks_per_sm);
/* The same for the whole grid (0 = no cap).  Any grid >= 1 CTA completes: a claimed task only waits on tasks
 * claimed earlier.  Errors: CONTEXT, BAD_N. */
int rna4r_set_max_blocks(rna4r_ctx *ctx, int blocks);

/*
 * rna4r_fold -- one fold (problem statement PAPER.md:45-54; wavefront PAPER.md:223-269).
 *   seq_dev       device uint8[n]: the bases S_1..S_n as ASCII bytes (read only).
 *   n             host int, 0 <= n <= 65534.
 *   score_out_dev device int32[1]: receives D(1,n) (-1 if seq holds an invalid byte).
 *   table_out_dev device or NULL: n*n elements row-major, entry [i-1][j-1] = D(i,j) for i <= j,
 *                 0 below the diagonal; element type given by table_dtype (RNA4R_TABLE_*;
 *                 pass RNA4R_TABLE_NONE with NULL).
 *   workspace_dev device scratch of >= rna4r_workspace_bytes(ctx, n, 1) bytes.
 * Errors: CONTEXT, NULL, BAD_N, DTYPE, WORKSPACE, CUDA (launch failure).
 */
int rna4r_fold(rna4r_ctx *ctx, const uint8_t *seq_dev, int n,
               int32_t *score_out_dev, void *table_out_dev, int table_dtype,
               void *workspace_dev, size_t workspace_bytes, void *stream);

/*
 * rna4r_fold_batch -- `count` independent folds in one call (BASELINE.json north_star; each fold
 * is PAPER.md:45-54).  Sequence t is seqs_dev[offsets_dev[t] .. offsets_dev[t+1]).
 *   seqs_dev       device uint8[offsets[count]]: concatenated bases.
 *   offsets_dev    device int64[count+1]: start offsets, offsets[0] = 0, non-decreasing.
 *   lens_host      HOST int32[count]: lens_host[t] = offsets[t+1]-offsets[t]; host memory so the
 *                  library can size and validate the work without a device synchronisation.  It is
 *                  consumed (copied) before the call returns.  The geometry of the work always
 *                  follows lens_host; a sequence whose device offsets disagree is not read and
 *                  scores -1 (RNA4R_STATUS_BAD_OFFSETS).
 *   scores_out_dev device int32[count]: D(1,n_t) per sequence (-1 for an invalid sequence).
 *   status_out_dev (rna4r_fold_batch_status only) device int32[count] or NULL: RNA4R_STATUS_* bits
 *                  per sequence, 0 = folded.
 *   workspace_dev  device scratch of >= rna4r_workspace_bytes_batch(ctx, lens_host, count).
 * Errors: CONTEXT, NULL, BAD_N, WORKSPACE, CUDA.
 */
int rna4r_fold_batch(rna4r_ctx *ctx, const uint8_t *seqs_dev, const int64_t *offsets_dev,
                     const int32_t *lens_host, int count, int32_t *scores_out_dev,
                     void *workspace_dev, size_t workspace_bytes, void *stream);
int rna4r_fold_batch_status(rna4r_ctx *ctx, const uint8_t *seqs_dev, const int64_t *offsets_dev,
                            const int32_t *lens_host, int count, int32_t *scores_out_dev,
                            int32_t *status_out_dev,
                            void *workspace_dev, size_t workspace_bytes, void *stream);

/*
 * rna4r_traceback -- one optimal structure (a maximum set of non-crossing complementary pairs) from a
 * finished table.  The paper stores arg-max indices beside the maxima (D*); this call
 * recovers the pairs from D alone by re-running eq. (1) along the optimal path: an interval
 * pairs its ends if b(S_i,S_j) = 1 and D(i,j) = 1 + D(i+1,j-1), else it splits at the smallest k in [i+1,j]
 * with D(i,j) = D(i,k-1) + D(k,j).  Deterministic; several structures may be optimal, this rule picks one.
 *   seq_dev        device uint8[n]: the bases (as given to rna4r_fold).
 *   table_dev      device n*n elements in the layout rna4r_fold writes (table_dtype INT16 or INT32).
 *   pairs_out_dev  device int32[n]: partner (0-based) of every base, -1 if unpaired.
 *   npairs_out_dev device int32[1]: number of pairs = D(1,n); -1 if the sequence holds an invalid byte or the
 *                  table is not a table of eq. (1) for this sequence.
 *   workspace_dev  device scratch of >= rna4r_traceback_workspace_bytes(ctx, n) bytes.
 * Enqueues only (no allocation, no synchronisation).  Errors: CONTEXT, NULL, BAD_N, DTYPE, WORKSPACE, CUDA.
 */
size_t rna4r_traceback_workspace_bytes(const rna4r_ctx *ctx, int n);
int rna4r_traceback(rna4r_ctx *ctx, const uint8_t *seq_dev, int n, const void *table_dev, int table_dtype,
                    int32_t *pairs_out_dev, int32_t *npairs_out_dev,
                    void *workspace_dev, size_t workspace_bytes, void *stream);

/*
 * Host-buffer variants (the end-to-end path): the sequence(s) are copied host->device into the
 * workspace, folded, the score(s) (and table) copied device->host, and `stream` is synchronised
 * before returning (once, at the end; no host allocation).  Host buffers should be pinned for full
 * copy bandwidth but need not be.
 * Workspace: rna4r_workspace_bytes_host(ctx, lens_host, count, table_dtype) = the device-side
 * requirement for these lengths plus the staging area (bases, offsets, scores, and -- count == 1,
 * table_dtype != RNA4R_TABLE_NONE -- the n*n table); 0 on error.
 *   table_out_host (rna4r_fold_host only): host n*n elements or NULL.
 */
size_t rna4r_workspace_bytes_host(const rna4r_ctx *ctx, const int32_t *lens_host, int count, int table_dtype);
int rna4r_fold_host(rna4r_ctx *ctx, const uint8_t *seq_host, int n,
                    int32_t *score_out_host, void *table_out_host, int table_dtype,
                    void *workspace_dev, size_t workspace_bytes, void *stream);
int rna4r_fold_batch_host(rna4r_ctx *ctx, const uint8_t *seqs_host, const int32_t *lens_host, int count,
                          int32_t *scores_out_host,
                          void *workspace_dev, size_t workspace_bytes, void *stream);

/* Number of kernel launches the most recent fold call enqueued (for accounting), or < 0. */
int rna4r_last_launch_count(const rna4r_ctx *ctx);

/*
 * Kernel timing for roofline accounting.  With timing enabled (on != 0) every fold call records a pair
 * of CUDA events on the launching stream around its dominant kernel -- the persistent fill kernel of
 * the TILED engine, or the whole sequence of per-diagonal launches of the DIAG engine (for a DIAG
 * batch: the last sequence).  rna4r_last_fill_kernel_ms waits for the second event and writes the
 * elapsed milliseconds to *ms_host.  Errors: CONTEXT, NULL, CUDA (also when nothing was recorded).
 */
int rna4r_enable_kernel_timing(rna4r_ctx *ctx, int on);
int rna4r_last_fill_kernel_ms(rna4r_ctx *ctx, float *ms_host);

/*
 * Wavefront trace (TILED engine; a profiling aid for the per-diagonal latency of step a7).  With
 * max_tiles > 0 the context allocates max_tiles * 64 bytes; every closure task of a later fold then
 * writes eight uint64 for its super-tile (index = order of the triangular enumeration, row-major
 * I <= J): %globaltimer ns at [0] task claimed, [1] static dependencies met, [2],[3] prologue loaded,
 * [4] closure warp 0 reached the final barrier, [5] record complete and flagged; [6] = I << 32 | J;
 * [7] = clock64 cycles of closure warp 0 in three 21-bit fields (fresh merge | cell wavefronts | barrier).
 * max_tiles = 0 frees the buffer and switches tracing off.  rna4r_trace_to_host synchronises the
 * device and copies `tiles` records to HOST memory.  Errors: CONTEXT, NULL, BAD_N, CUDA.
 */
int rna4r_set_trace(rna4r_ctx *ctx, int max_tiles);
int rna4r_trace_to_host(rna4r_ctx *ctx, uint64_t *dst_host, int tiles);

/*
 * Measured ceiling of the lookup sequence (a profiling aid for the roofline denominator).
 * Runs, from every SM and free of bank conflicts, the instruction sequence of one table lookup of eq. (3)
 * as the fill kernel issues it, and times it with CUDA events on `stream` (synchronises):
 *   variant 0 (context q = 8):  add, address, 1-byte shared-memory gather, add-max; operands in registers;
 *   variant 1 (context q = 8):  the bulk product's inner loop (operand words loaded from shared memory);
 *   variant 2 (context q = 10): variant 0 on the ternary-indexed table of 3^9 entries; operands in registers.
 *   iters           loop trips per thread, 1..16000 (16 lookups per trip; variant 1: 128 per trip).
 *   blocks_per_sm   CTAs of 256 threads per SM (0 = as many as fit).
 *   workspace_dev   device scratch, >= 256 bytes.
 *   ms_host, lookups_host   HOST outputs: elapsed milliseconds and the number of lookups executed.
 * Errors: CONTEXT, NULL, BAD_N, ENGINE (variant does not match the context's q), CUDA.
 */
int rna4r_microbench_lookups(rna4r_ctx *ctx, int variant, int iters, int blocks_per_sm, void *workspace_dev,
                             void *stream, float *ms_host, double *lookups_host);

/*
 * A fold that allocates nothing and takes no workspace, for callers that cannot call cudaMalloc (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it).  The same fill as rna4r_fold with
 * RNA4R_ENGINE_TILED, score only (D(1,n) of eq. (1)), whatever engine the context is set to; its
 * scratch (plan, flags, super-tile records, bulk maxima) is a static device array inside the library of
 * RNA4R_STATIC_SCRATCH_BYTES, which every GPU that loads the library holds until the process exits.
 *
 *   rna4r_fold_static_setup   once per device (any context of that device, q <= 11; repeat it for every q used, it
 *                             also warms that q's kernels up): looks the array's device address up, runs one
 *                             100-base fold out of the array's tail on `stream` and synchronises that stream.  Not
 *                             for use under graph capture.  Errors: CONTEXT, ENGINE (q = 12), DEVICE, CUDA.
 *   rna4r_fold_static_max_n   largest n whose scratch fits the array for the context's q (1567 at q = 2, 1951 at q = 4,
 *                             2239 at q = 8, 2375 at q = 11), or a
 *                             negative error code (CONTEXT, ENGINE).
 *   rna4r_fold_static         seq_dev: DEVICE, n ASCII bases (not modified; may be NULL if n == 0); score_out_dev:
 *                             DEVICE int32, written when the stream work completes (-1 for a byte that is not a base,
 *                             reading g4).  Enqueues on `stream` and returns; calls no cudaMalloc / cudaFree or
 *                             allocating routine.  Errors: CONTEXT, ENGINE (q = 12), NULL, BAD_N (n < 0 or
 *                             n > rna4r_fold_static_max_n: nothing is enqueued), SETUP (rna4r_fold_static_setup has
 *                             not run on this device in this process), CUDA.
 *
 * Every call on a device shares the one array, whatever its context or stream, and the array keeps the last
 * call's contents: each fold zeroes the part that has to start at zero itself, but two calls whose GPU work
 * overlaps (different streams without an ordering between them, or two host threads) race.  Order them on one
 * stream or with events.  The process-wide setup state is not guarded against concurrent setup calls.
 */
#define RNA4R_STATIC_SCRATCH_BYTES (8u << 20)
int rna4r_fold_static_setup(rna4r_ctx *ctx, void *stream);
int rna4r_fold_static_max_n(const rna4r_ctx *ctx);
int rna4r_fold_static(rna4r_ctx *ctx, const uint8_t *seq_dev, int n, int32_t *score_out_dev, void *stream);

/* cudaError_t of the most recent failing CUDA call on this context (0 if none). */
int rna4r_last_cuda_error(const rna4r_ctx *ctx);

/* Static string for an error code. */
const char *rna4r_strerror(int code);

/* Library / build identification, e.g. "rna4r 0.1 sm_100a". */
const char *rna4r_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RNA4R_H */
