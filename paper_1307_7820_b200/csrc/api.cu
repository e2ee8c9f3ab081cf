// api.cu -- the C ABI of librna4r.so (include/rna4r.h): context, workspace planning, dispatch.
#include <new>
#include "common.cuh"
#include "rtable.cuh"
#include "diag_engine.cuh"
#include "tiled_engine.cuh"
#include "smem_engine.cuh"
#include "compare_engines.cuh"
#include "traceback.cuh"
#include "microbench.cuh"


namespace {

constexpr int kDelta = 0;   // 0: the tiled engine picks the product-stage span from the problem size

inline bool ctx_ok(const rna4r_ctx *c) { return c && c->magic == RNA4R_MAGIC; }

template <typename F>
auto dispatch_q_smem(int q, F &&f) -> decltype(f(std::integral_constant<int, 8>{}))
{
    switch (q) {
    case 4: return f(std::integral_constant<int, 4>{});
    case 5: return f(std::integral_constant<int, 5>{});
    case 6: return f(std::integral_constant<int, 6>{});
    case 7: return f(std::integral_constant<int, 7>{});
    default: return f(std::integral_constant<int, 8>{});
    }
}

template <typename F>
auto dispatch_q(int q, F &&f) -> decltype(f(std::integral_constant<int, 8>{}))
{
    switch (q) {
    case 2: return f(std::integral_constant<int, 2>{});
    case 3: return f(std::integral_constant<int, 3>{});
    case 4: return f(std::integral_constant<int, 4>{});
    case 5: return f(std::integral_constant<int, 5>{});
    case 6: return f(std::integral_constant<int, 6>{});
    case 7: return f(std::integral_constant<int, 7>{});
    case 8: return f(std::integral_constant<int, 8>{});
    case 9: return f(std::integral_constant<int, 9>{});
    case 10: return f(std::integral_constant<int, 10>{});
    default: return f(std::integral_constant<int, 11>{});
    }
}

// largest n the tagged 32-bit words of the tiled engine can hold: the value field is 16 bits for every q
// (tiled::Cfg: ISHIFT = 16), anchor sums + q < 2^16 with D <= n/2, so the ABI's limit n <= 65534 (int16 table) is the only one
inline int tiled_max_n(int q)
{
    (void)q;
    return 65534;
}

size_t tiled_ws(const rna4r_ctx *ctx, const int32_t *lens, int count, int n_single)
{
    return dispatch_q(ctx->q, [&](auto Q) { return tiled::workspace_bytes_q<decltype(Q)::value>(kDelta, lens, count, n_single); });
}

// RNA4R_ENGINE_SMEM: q = 4..8, and the sequence's state has to fit one CTA's shared memory (n <= 704 at q = 8)
inline bool smem_q_ok(int q) { return q >= 4 && q <= 8; }
inline int smem_max_n(int q)
{
    switch (q) {
    case 4: return smemseq::max_n<4>();
    case 5: return smemseq::max_n<5>();
    case 6: return smemseq::max_n<6>();
    case 7: return smemseq::max_n<7>();
    case 8: return smemseq::max_n<8>();
    default: return -1;
    }
}

// the engines that fold one sequence per call (the comparison engines): workspace of one fold, and the enqueue
inline bool per_sequence_engine(int e) { return e == RNA4R_ENGINE_DIAG || e == RNA4R_ENGINE_PAPER_TILE || e == RNA4R_ENGINE_MAXPLUS; }
size_t single_ws(const rna4r_ctx *ctx, int n)
{
    if (ctx->engine == RNA4R_ENGINE_PAPER_TILE) return cmpeng::pt_layout(nullptr, n, ctx->q).bytes;
    if (ctx->engine == RNA4R_ENGINE_MAXPLUS) return cmpeng::mp_layout(nullptr, n).bytes;
    return diag_ws_layout(nullptr, n).bytes;
}
int single_enqueue(rna4r_ctx *ctx, const uint8_t *seq_dev, const int64_t *offset_dev, int n, int32_t *score_dev, int32_t *status_dev,
                   void *table_out, int table_dtype, void *ws, cudaStream_t st)
{
    if (ctx->engine == RNA4R_ENGINE_PAPER_TILE)
        return cmpeng::pt_fold_enqueue(ctx, seq_dev, offset_dev, n, score_dev, status_dev, table_out, table_dtype, ws, st);
    if (ctx->engine == RNA4R_ENGINE_MAXPLUS)
        return cmpeng::mp_fold_enqueue(ctx, seq_dev, offset_dev, n, score_dev, status_dev, table_out, table_dtype, ws, st);
    return diag_fold_enqueue(ctx, seq_dev, offset_dev, n, score_dev, status_dev, table_out, table_dtype, ws, st);
}

size_t engine_ws(const rna4r_ctx *ctx, const int32_t *lens, int count, int n_single)
{
    if (ctx->engine == RNA4R_ENGINE_SMEM) return smemseq::workspace_bytes(count);
    if (ctx->engine == RNA4R_ENGINE_TILED)      // AUTO may split a batch: the tiled engine's area, then the SMEM engine's
        return align_up(tiled_ws(ctx, lens, count, n_single), 256) + (ctx->engine_auto ? smemseq::workspace_bytes(count) : 0);
    // per-sequence engines: sequences of a batch are folded one after another, each in its own slice
    size_t total = 0;
    for (int t = 0; t < count; ++t) total += single_ws(ctx, lens ? lens[t] : n_single);
    return total;
}

int check_n(const rna4r_ctx *ctx, int n)
{
    if (n < 0 || n > 65534) return RNA4R_ERR_BAD_N;
    if (ctx->engine == RNA4R_ENGINE_TILED && n > tiled_max_n(ctx->q)) return RNA4R_ERR_BAD_N;
    if (ctx->engine == RNA4R_ENGINE_SMEM && n > smem_max_n(ctx->q)) return RNA4R_ERR_BAD_N;
    return RNA4R_OK;
}

}  // namespace

extern "C" {

const char *rna4r_version(void) { return "rna4r 0.1 sm_100a"; }

const char *rna4r_strerror(int code)
{
    switch (code) {
    case RNA4R_OK: return "ok";
    case RNA4R_ERR_BAD_Q: return "q outside 2..12";
    case RNA4R_ERR_NULL: return "required pointer is NULL";
    case RNA4R_ERR_BAD_N: return "bad n or count (negative, or too large for this engine and q)";
    case RNA4R_ERR_WORKSPACE: return "workspace too small";
    case RNA4R_ERR_CONTEXT: return "invalid context";
    case RNA4R_ERR_CUDA: return "CUDA runtime error";
    case RNA4R_ERR_DEVICE: return "no sm_100 CUDA device (there is no CPU fallback)";
    case RNA4R_ERR_DTYPE: return "bad table dtype";
    case RNA4R_ERR_ENGINE: return "unknown engine, or engine does not support this q";
    case RNA4R_ERR_SETUP: return "rna4r_fold_static before rna4r_fold_static_setup on this device";
    default: return "unknown error code";
    }
}

int rna4r_prepare(int q, int device, void *stream, rna4r_ctx **out)
{
    if (!out) return RNA4R_ERR_NULL;
    *out = nullptr;
    if (q < 2 || q > 12) return RNA4R_ERR_BAD_Q;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0 || device < 0 || device >= ndev) {
        cudaGetLastError();
        return RNA4R_ERR_DEVICE;
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return RNA4R_ERR_DEVICE;
    if (prop.major != 10 || prop.minor != 0) return RNA4R_ERR_DEVICE;   // the library holds sm_100a code only; no fallback path exists
    rna4r_ctx *ctx = new (std::nothrow) rna4r_ctx();
    if (!ctx) return RNA4R_ERR_CUDA;
    ctx->magic = RNA4R_MAGIC; ctx->q = q; ctx->device = device;
    ctx->engine = (q <= 11) ? RNA4R_ENGINE_TILED : RNA4R_ENGINE_DIAG;
    ctx->sm_count = prop.multiProcessorCount;
    ctx->R = ctx->Rc = ctx->Rt = nullptr;
    ctx->last_launches = 0; ctx->last_cuda_error = 0; ctx->tiled_blocks_per_sm = 0; ctx->max_blocks_per_sm = 0; ctx->max_blocks = 0;
    ctx->timing = 0; ctx->timing_valid = 0; ctx->ev0 = ctx->ev1 = nullptr;
    ctx->trace = nullptr; ctx->trace_tiles = 0;
    ctx->engine_auto = 1; ctx->order_host = nullptr; ctx->order_cap = 0; ctx->route_host = nullptr; ctx->route_cap = 0;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t N = (size_t)1 << q, M = (size_t)1 << (q - 1);
    auto fail = [&](cudaError_t e) { ctx->last_cuda_error = (int)e; cudaFree(ctx->R); cudaFree(ctx->Rc); cudaFree(ctx->Rt); delete ctx; return RNA4R_ERR_CUDA; };
    cudaError_t e;
    if ((e = cudaSetDevice(device)) != cudaSuccess) return fail(e);
    if ((e = cudaMalloc(&ctx->R, N * N)) != cudaSuccess) return fail(e);
    if ((e = cudaMalloc(&ctx->Rc, M * M < 16 ? 16 : M * M)) != cudaSuccess) return fail(e);
    uint32_t tern = 0;                                   // 3^(q-1) entries, built for the q that use them (tiled::Cfg::TERN)
    if (q >= RNA4R_TERN_MIN_Q && q <= 11) { tern = 1; for (int k = 1; k < q; ++k) tern *= 3u; }
    if (tern && (e = cudaMalloc(&ctx->Rt, (tern + 15u) & ~15u)) != cudaSuccess) return fail(e);
    {
        const size_t total = N * N;
        const int cap = ctx->sm_count * 16;
        int blocks = (int)((total + 255) / 256); if (blocks > cap) blocks = cap;
        rna4r_build_rtable_kernel<<<blocks, 256, 0, st>>>(q, ctx->R);
        const size_t tc = M * M;
        blocks = (int)((tc + 255) / 256); if (blocks > cap) blocks = cap;
        rna4r_build_compact_kernel<<<blocks, 256, 0, st>>>(q, ctx->R, ctx->Rc);
        ctx->last_launches = 2;
        if (tern) {
            if ((e = cudaMemsetAsync(ctx->Rt, 0, (tern + 15u) & ~15u, st)) != cudaSuccess) return fail(e);
            rna4r_build_ternary_kernel<<<(int)((tern + 255u) / 256u), 256, 0, st>>>(q, tern, ctx->Rt);
            ctx->last_launches = 3;
        }
        if ((e = cudaGetLastError()) != cudaSuccess) return fail(e);
    }
    *out = ctx;
    return RNA4R_OK;
}

int rna4r_destroy(rna4r_ctx *ctx)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    cudaFree(ctx->R); cudaFree(ctx->Rc); cudaFree(ctx->Rt);
    cudaFree(ctx->trace);
    if (ctx->ev0) cudaEventDestroy(ctx->ev0);
    if (ctx->ev1) cudaEventDestroy(ctx->ev1);
    delete[] ctx->order_host;
    delete[] ctx->route_host;
    ctx->magic = 0;
    delete ctx;
    return RNA4R_OK;
}

int rna4r_q(const rna4r_ctx *ctx) { return ctx_ok(ctx) ? ctx->q : RNA4R_ERR_CONTEXT; }
const uint8_t *rna4r_table(const rna4r_ctx *ctx) { return ctx_ok(ctx) ? ctx->R : nullptr; }
const uint8_t *rna4r_table_compact(const rna4r_ctx *ctx) { return ctx_ok(ctx) ? ctx->Rc : nullptr; }
int rna4r_engine(const rna4r_ctx *ctx) { return ctx_ok(ctx) ? ctx->engine : RNA4R_ERR_CONTEXT; }
int rna4r_smem_max_n(const rna4r_ctx *ctx) { return ctx_ok(ctx) ? smem_max_n(ctx->q) : RNA4R_ERR_CONTEXT; }
int rna4r_last_launch_count(const rna4r_ctx *ctx) { return ctx_ok(ctx) ? ctx->last_launches : RNA4R_ERR_CONTEXT; }
int rna4r_last_cuda_error(const rna4r_ctx *ctx) { return ctx_ok(ctx) ? ctx->last_cuda_error : RNA4R_ERR_CONTEXT; }

int rna4r_table_to_host(rna4r_ctx *ctx, uint8_t *dst_host, int compact)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (!dst_host) return RNA4R_ERR_NULL;
    RNA4R_CUDA(ctx, cudaSetDevice(ctx->device));
    RNA4R_CUDA(ctx, cudaDeviceSynchronize());
    if (compact < 0 || compact > 2) return RNA4R_ERR_BAD_N;
    if (compact == 2) {                                  // the ternary-indexed table, 3^(q-1) bytes (q = 9..11 only)
        if (!ctx->Rt) return RNA4R_ERR_ENGINE;
        size_t entries = 1;
        for (int k = 1; k < ctx->q; ++k) entries *= 3;
        RNA4R_CUDA(ctx, cudaMemcpy(dst_host, ctx->Rt, entries, cudaMemcpyDeviceToHost));
        return RNA4R_OK;
    }
    const size_t side = (size_t)1 << (compact ? ctx->q - 1 : ctx->q);
    RNA4R_CUDA(ctx, cudaMemcpy(dst_host, compact ? ctx->Rc : ctx->R, side * side, cudaMemcpyDeviceToHost));
    return RNA4R_OK;
}

int rna4r_set_trace(rna4r_ctx *ctx, int max_tiles)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    RNA4R_CUDA(ctx, cudaSetDevice(ctx->device));
    RNA4R_CUDA(ctx, cudaDeviceSynchronize());
    cudaFree(ctx->trace);
    ctx->trace = nullptr; ctx->trace_tiles = 0;
    if (max_tiles > 0) {
        RNA4R_CUDA(ctx, cudaMalloc(&ctx->trace, (size_t)max_tiles * 8 * RNA4R_TRACE_WORDS));
        RNA4R_CUDA(ctx, cudaMemset(ctx->trace, 0, (size_t)max_tiles * 8 * RNA4R_TRACE_WORDS));
        ctx->trace_tiles = max_tiles;
    }
    return RNA4R_OK;
}

int rna4r_trace_to_host(rna4r_ctx *ctx, uint64_t *dst_host, int tiles)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (!dst_host) return RNA4R_ERR_NULL;
    if (!ctx->trace || tiles < 0 || tiles > ctx->trace_tiles) return RNA4R_ERR_BAD_N;
    RNA4R_CUDA(ctx, cudaSetDevice(ctx->device));
    RNA4R_CUDA(ctx, cudaDeviceSynchronize());
    RNA4R_CUDA(ctx, cudaMemcpy(dst_host, ctx->trace, (size_t)tiles * 8 * RNA4R_TRACE_WORDS, cudaMemcpyDeviceToHost));
    return RNA4R_OK;
}

int rna4r_enable_kernel_timing(rna4r_ctx *ctx, int on)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    RNA4R_CUDA(ctx, cudaSetDevice(ctx->device));
    if (on && !ctx->ev0) {
        RNA4R_CUDA(ctx, cudaEventCreate(&ctx->ev0));
        RNA4R_CUDA(ctx, cudaEventCreate(&ctx->ev1));
    }
    ctx->timing = on ? 1 : 0;
    ctx->timing_valid = 0;
    return RNA4R_OK;
}

int rna4r_last_fill_kernel_ms(rna4r_ctx *ctx, float *ms_host)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (!ms_host) return RNA4R_ERR_NULL;
    if (!ctx->timing_valid) { ctx->last_cuda_error = 0; return RNA4R_ERR_CUDA; }
    RNA4R_CUDA(ctx, cudaEventSynchronize(ctx->ev1));
    RNA4R_CUDA(ctx, cudaEventElapsedTime(ms_host, ctx->ev0, ctx->ev1));
    return RNA4R_OK;
}

int rna4r_set_engine(rna4r_ctx *ctx, int engine)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    const int is_auto = engine == RNA4R_ENGINE_AUTO;
    if (is_auto) engine = (ctx->q <= 11) ? RNA4R_ENGINE_TILED : RNA4R_ENGINE_DIAG;
    if (engine != RNA4R_ENGINE_TILED && engine != RNA4R_ENGINE_SMEM && !per_sequence_engine(engine)) return RNA4R_ERR_ENGINE;
    if (engine == RNA4R_ENGINE_TILED && ctx->q > 11) return RNA4R_ERR_ENGINE;
    if (engine == RNA4R_ENGINE_SMEM && !smem_q_ok(ctx->q)) return RNA4R_ERR_ENGINE;
    ctx->engine = engine;
    ctx->engine_auto = is_auto;
    return RNA4R_OK;
}

int rna4r_set_max_blocks_per_sm(rna4r_ctx *ctx, int blocks_per_sm)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (blocks_per_sm < 0) return RNA4R_ERR_BAD_N;
    ctx->max_blocks_per_sm = blocks_per_sm;
    return RNA4R_OK;
}

int rna4r_set_max_blocks(rna4r_ctx *ctx, int blocks)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (blocks < 0) return RNA4R_ERR_BAD_N;
    ctx->max_blocks = blocks;
    return RNA4R_OK;
}

static size_t host_staging_bytes(size_t total_bases, int count, size_t table_bytes);

size_t rna4r_workspace_bytes(const rna4r_ctx *ctx, int n_max, int count, int flags)
{
    if (!ctx_ok(ctx) || n_max < 0 || count < 0 || n_max > 65534) return 0;
    if (flags & ~(RNA4R_WS_HOST_STAGING | RNA4R_WS_HOST_TABLE16 | RNA4R_WS_HOST_TABLE32)) return 0;
    size_t core = 256;
    if (count > 0) {
        // every sequence at n_max: per-sequence cost is monotone in n
        if (ctx->engine == RNA4R_ENGINE_TILED) core = (size_t)count * tiled_ws(ctx, nullptr, 1, n_max) + smemseq::workspace_bytes(count);
        else if (ctx->engine == RNA4R_ENGINE_SMEM) core = smemseq::workspace_bytes(count);
        else core = (size_t)count * single_ws(ctx, n_max);
    }
    if (!(flags & (RNA4R_WS_HOST_STAGING | RNA4R_WS_HOST_TABLE16 | RNA4R_WS_HOST_TABLE32))) return core;
    size_t table_bytes = 0;
    if (count == 1 && (flags & RNA4R_WS_HOST_TABLE32)) table_bytes = (size_t)n_max * n_max * 4;
    else if (count == 1 && (flags & RNA4R_WS_HOST_TABLE16)) table_bytes = (size_t)n_max * n_max * 2;
    return align_up(core, 256) + host_staging_bytes((size_t)count * n_max, count, table_bytes);
}

size_t rna4r_workspace_bytes_batch(const rna4r_ctx *ctx, const int32_t *lens_host, int count)
{
    if (!ctx_ok(ctx) || count < 0 || (!lens_host && count > 0)) return 0;
    if (count == 0) return 256;
    for (int t = 0; t < count; ++t) if (lens_host[t] < 0 || lens_host[t] > 65534) return 0;
    return engine_ws(ctx, lens_host, count, 0);
}

int rna4r_fold(rna4r_ctx *ctx, const uint8_t *seq_dev, int n, int32_t *score_out_dev,
               void *table_out_dev, int table_dtype, void *workspace_dev, size_t workspace_bytes, void *stream)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (!score_out_dev || !workspace_dev || (!seq_dev && n > 0)) return RNA4R_ERR_NULL;
    int rc = check_n(ctx, n);
    if (rc != RNA4R_OK) return rc;
    if (table_dtype != RNA4R_TABLE_NONE && table_dtype != RNA4R_TABLE_INT16 && table_dtype != RNA4R_TABLE_INT32) return RNA4R_ERR_DTYPE;
    if ((table_dtype == RNA4R_TABLE_NONE) != (table_out_dev == nullptr)) return table_out_dev ? RNA4R_ERR_DTYPE : RNA4R_ERR_NULL;
    if (workspace_bytes < engine_ws(ctx, nullptr, 1, n)) return RNA4R_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    RNA4R_CUDA(ctx, cudaSetDevice(ctx->device));
    if (ctx->engine == RNA4R_ENGINE_DIAG)
        return diag_fold_enqueue(ctx, seq_dev, nullptr, n, score_out_dev, nullptr, table_out_dev, table_dtype, workspace_dev, st);
    if (table_out_dev && n > 0) {
        const size_t es = table_dtype == RNA4R_TABLE_INT16 ? 2 : 4;
        RNA4R_CUDA(ctx, cudaMemsetAsync(table_out_dev, 0, (size_t)n * n * es, st));   // zeros below the diagonal
    }
    if (per_sequence_engine(ctx->engine))      // PAPER_TILE / MAXPLUS (DIAG returned above: it writes the whole table itself)
        return single_enqueue(ctx, seq_dev, nullptr, n, score_out_dev, nullptr, table_out_dev, table_dtype, workspace_dev, st);
    if (ctx->engine == RNA4R_ENGINE_SMEM)
        return dispatch_q_smem(ctx->q, [&](auto Q) {
            return smemseq::enqueue_q<decltype(Q)::value>(ctx, seq_dev, nullptr, nullptr, 1, n, score_out_dev, nullptr, table_out_dev,
                                                          table_dtype, workspace_dev, st);
        });
    return dispatch_q(ctx->q, [&](auto Q) {
        return tiled::enqueue_q<decltype(Q)::value>(ctx, kDelta, seq_dev, nullptr, nullptr, 1, n, score_out_dev, nullptr,
                                                    table_out_dev, table_dtype, workspace_dev, st);
    });
}

int rna4r_fold_batch(rna4r_ctx *ctx, const uint8_t *seqs_dev, const int64_t *offsets_dev, const int32_t *lens_host,
                     int count, int32_t *scores_out_dev, void *workspace_dev, size_t workspace_bytes, void *stream)
{
    return rna4r_fold_batch_status(ctx, seqs_dev, offsets_dev, lens_host, count, scores_out_dev, nullptr, workspace_dev,
                                   workspace_bytes, stream);
}

int rna4r_fold_batch_status(rna4r_ctx *ctx, const uint8_t *seqs_dev, const int64_t *offsets_dev, const int32_t *lens_host,
                            int count, int32_t *scores_out_dev, int32_t *status_out_dev, void *workspace_dev,
                            size_t workspace_bytes, void *stream)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (count < 0) return RNA4R_ERR_BAD_N;
    if (count == 0) { ctx->last_launches = 0; return RNA4R_OK; }
    if (!offsets_dev || !lens_host || !scores_out_dev || !workspace_dev) return RNA4R_ERR_NULL;
    size_t total_bases = 0;
    for (int t = 0; t < count; ++t) {
        int rc = check_n(ctx, lens_host[t]);
        if (rc != RNA4R_OK) return rc;
        total_bases += (size_t)lens_host[t];
    }
    if (!seqs_dev && total_bases > 0) return RNA4R_ERR_NULL;
    if (workspace_bytes < engine_ws(ctx, lens_host, count, 0)) return RNA4R_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    RNA4R_CUDA(ctx, cudaSetDevice(ctx->device));
    if (per_sequence_engine(ctx->engine)) {
        size_t ws_off = 0;            // sequence t starts at offsets_dev[t] (read on the device)
        int launches = 0;
        for (int t = 0; t < count; ++t) {
            int rc = single_enqueue(ctx, seqs_dev, offsets_dev + t, lens_host[t], scores_out_dev + t,
                                    status_out_dev ? status_out_dev + t : nullptr, nullptr, RNA4R_TABLE_NONE,
                                    (char *)workspace_dev + ws_off, st);
            if (rc != RNA4R_OK) return rc;
            launches += ctx->last_launches;
            ws_off += single_ws(ctx, lens_host[t]);
        }
        ctx->last_launches = launches;
        return RNA4R_OK;
    }
    // AUTO: sequences whose state fits one CTA's shared memory go to the CTA-per-sequence engine, the
    // longer ones of the same batch to the tiled engine (indexed through a map: nothing is copied or reordered).
    if (ctx->engine == RNA4R_ENGINE_SMEM)
        return dispatch_q_smem(ctx->q, [&](auto Q) {
            return smemseq::enqueue_q<decltype(Q)::value>(ctx, seqs_dev, offsets_dev, lens_host, count, 0, scores_out_dev,
                                                          status_out_dev, nullptr, RNA4R_TABLE_NONE, workspace_dev, st);
        });
    if (ctx->engine_auto && smem_q_ok(ctx->q)) {
        const int lim = smem_max_n(ctx->q);
        int n_long = 0;
        for (int t = 0; t < count; ++t) n_long += lens_host[t] > lim;
        if (n_long < count) {
            const size_t smem_off = n_long ? align_up(tiled_ws(ctx, lens_host, count, 0), 256) : 0;
            int launches = 0;
            if (n_long) {
                if (count > ctx->route_cap) {
                    int32_t *nb = new (std::nothrow) int32_t[2 * (size_t)count];
                    if (!nb) return RNA4R_ERR_CUDA;
                    delete[] ctx->route_host;
                    ctx->route_host = nb; ctx->route_cap = count;
                }
                int32_t *idx = ctx->route_host, *len = idx + count;
                for (int t = 0, k = 0; t < count; ++t) if (lens_host[t] > lim) { idx[k] = t; len[k++] = lens_host[t]; }
                int rc = dispatch_q(ctx->q, [&](auto Q) {
                    return tiled::enqueue_q<decltype(Q)::value>(ctx, kDelta, seqs_dev, offsets_dev, len, n_long, 0, scores_out_dev,
                                                                status_out_dev, nullptr, RNA4R_TABLE_NONE, workspace_dev, st, idx);
                });
                if (rc != RNA4R_OK) return rc;
                launches = ctx->last_launches;
            }
            int rc = dispatch_q_smem(ctx->q, [&](auto Q) {
                return smemseq::enqueue_q<decltype(Q)::value>(ctx, seqs_dev, offsets_dev, lens_host, count, 0, scores_out_dev,
                                                              status_out_dev, nullptr, RNA4R_TABLE_NONE, (char *)workspace_dev + smem_off,
                                                              st, true);
            });
            ctx->last_launches += launches;
            return rc;
        }
    }
    return dispatch_q(ctx->q, [&](auto Q) {
        return tiled::enqueue_q<decltype(Q)::value>(ctx, kDelta, seqs_dev, offsets_dev, lens_host, count, 0, scores_out_dev,
                                                    status_out_dev, nullptr, RNA4R_TABLE_NONE, workspace_dev, st);
    });
}

// ---- measured ceiling of the lookup sequence (profiling aid; microbench.cuh) ------------------------------------
int rna4r_microbench_lookups(rna4r_ctx *ctx, int variant, int iters, int blocks_per_sm, void *workspace_dev, void *stream,
                             float *ms_host, double *lookups_host)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (!workspace_dev || !ms_host || !lookups_host) return RNA4R_ERR_NULL;
    if (iters < 1 || iters > 16000) return RNA4R_ERR_BAD_N;
    cudaStream_t st = (cudaStream_t)stream;
    RNA4R_CUDA(ctx, cudaSetDevice(ctx->device));
    uint32_t *sink = (uint32_t *)workspace_dev;
    if (variant == 0 && ctx->q == 8) return microbench::run<8, 0>(ctx, iters, blocks_per_sm, sink, st, ms_host, lookups_host);
    if (variant == 1 && ctx->q == 8) return microbench::run<8, 1>(ctx, iters, blocks_per_sm, sink, st, ms_host, lookups_host);
    if (variant == 2 && ctx->q == 10) return microbench::run<10, 0>(ctx, iters, blocks_per_sm, sink, st, ms_host, lookups_host);
    return RNA4R_ERR_ENGINE;
}

// ---- traceback: one optimal structure from a finished table ------------------------
size_t rna4r_traceback_workspace_bytes(const rna4r_ctx *ctx, int n)
{
    if (!ctx_ok(ctx) || n < 0 || n > 65534) return 0;
    return traceback::workspace_bytes(n);
}

int rna4r_traceback(rna4r_ctx *ctx, const uint8_t *seq_dev, int n, const void *table_dev, int table_dtype,
                    int32_t *pairs_out_dev, int32_t *npairs_out_dev, void *workspace_dev, size_t workspace_bytes, void *stream)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (n < 0 || n > 65534) return RNA4R_ERR_BAD_N;
    if (!npairs_out_dev || !workspace_dev || (n > 0 && (!seq_dev || !table_dev || !pairs_out_dev))) return RNA4R_ERR_NULL;
    if (table_dtype != RNA4R_TABLE_INT16 && table_dtype != RNA4R_TABLE_INT32) return RNA4R_ERR_DTYPE;
    if (workspace_bytes < traceback::workspace_bytes(n)) return RNA4R_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    RNA4R_CUDA(ctx, cudaSetDevice(ctx->device));
    traceback::Queue *q = (traceback::Queue *)workspace_dev;
    unsigned long long *slots = (unsigned long long *)((char *)workspace_dev + 256);
    const int nslots = 2 * n + 64;
    traceback::init_kernel<<<(nslots + 255) / 256, 256, 0, st>>>(q, slots, nslots, pairs_out_dev, n);
    if (n >= 2) {
        int blocks = ctx->sm_count;
        if (blocks > (n + 63) / 64) blocks = (n + 63) / 64;       // small folds have few branches
        if (table_dtype == RNA4R_TABLE_INT16)
            traceback::walk_kernel<int16_t><<<blocks, 256, 0, st>>>(seq_dev, n, (const int16_t *)table_dev, q, slots, pairs_out_dev);
        else
            traceback::walk_kernel<int32_t><<<blocks, 256, 0, st>>>(seq_dev, n, (const int32_t *)table_dev, q, slots, pairs_out_dev);
    }
    traceback::finish_kernel<<<1, 32, 0, st>>>(q, npairs_out_dev);
    RNA4R_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = n >= 2 ? 3 : 2;
    return RNA4R_OK;
}

// ---- host-buffer variants: staging area at the END of the workspace --------------------------------
// offsets[0..count] = exclusive prefix sum of lens[0..count) (one block; count is at most a few 10^5)
__global__ void rna4r_offsets_from_lens_kernel(const int32_t *__restrict__ lens, int count, int64_t *__restrict__ offsets)
{
    __shared__ long long part[1024];
    const int tid = threadIdx.x, nth = blockDim.x;
    const int per = (count + nth - 1) / nth;
    const int lo = min(tid * per, count), hi = min(lo + per, count);
    long long sum = 0;
    for (int t = lo; t < hi; ++t) sum += lens[t];
    part[tid] = sum;
    __syncthreads();
    for (int d = 1; d < nth; d <<= 1) {          // inclusive scan of the per-thread sums
        const long long v = (tid >= d) ? part[tid - d] : 0;
        __syncthreads();
        part[tid] += v;
        __syncthreads();
    }
    long long run = part[tid] - sum;
    for (int t = lo; t < hi; ++t) { offsets[t] = run; run += lens[t]; }
    if (tid == nth - 1) offsets[count] = part[nth - 1];
}

static size_t host_staging_bytes(size_t total_bases, int count, size_t table_bytes)
{
    return align_up(total_bases + 16, 256) + align_up((size_t)(count + 1) * 8, 256) + align_up((size_t)count * 4 + 16, 256) + align_up(table_bytes, 256);
}

size_t rna4r_workspace_bytes_host(const rna4r_ctx *ctx, const int32_t *lens_host, int count, int table_dtype)
{
    if (!ctx_ok(ctx) || count < 0 || (!lens_host && count > 0)) return 0;
    size_t total_bases = 0;
    for (int t = 0; t < count; ++t) { if (lens_host[t] < 0 || lens_host[t] > 65534) return 0; total_bases += (size_t)lens_host[t]; }
    size_t table_bytes = 0;
    if (table_dtype != RNA4R_TABLE_NONE && count == 1)
        table_bytes = (size_t)lens_host[0] * lens_host[0] * (table_dtype == RNA4R_TABLE_INT16 ? 2 : 4);
    const size_t core = count ? engine_ws(ctx, lens_host, count, 0) : 256;
    return align_up(core, 256) + host_staging_bytes(total_bases, count, table_bytes);
}

int rna4r_fold_host(rna4r_ctx *ctx, const uint8_t *seq_host, int n, int32_t *score_out_host,
                    void *table_out_host, int table_dtype, void *workspace_dev, size_t workspace_bytes, void *stream)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (!score_out_host || !workspace_dev || (!seq_host && n > 0)) return RNA4R_ERR_NULL;
    int rc = check_n(ctx, n);
    if (rc != RNA4R_OK) return rc;
    if (table_dtype != RNA4R_TABLE_NONE && table_dtype != RNA4R_TABLE_INT16 && table_dtype != RNA4R_TABLE_INT32) return RNA4R_ERR_DTYPE;
    if ((table_dtype == RNA4R_TABLE_NONE) != (table_out_host == nullptr)) return table_out_host ? RNA4R_ERR_DTYPE : RNA4R_ERR_NULL;
    const int32_t len1 = n;
    if (workspace_bytes < rna4r_workspace_bytes_host(ctx, &len1, 1, table_dtype)) return RNA4R_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    RNA4R_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t core = align_up(engine_ws(ctx, nullptr, 1, n), 256);
    char *stg = (char *)workspace_dev + core;
    uint8_t *seq_dev = (uint8_t *)stg; stg += align_up((size_t)n + 16, 256);
    stg += align_up(2 * 8, 256);
    int32_t *score_dev = (int32_t *)stg; stg += align_up(4 + 16, 256);
    void *table_dev = table_out_host ? (void *)stg : nullptr;
    const size_t table_bytes = table_out_host ? (size_t)n * n * (table_dtype == RNA4R_TABLE_INT16 ? 2 : 4) : 0;
    if (n > 0) RNA4R_CUDA(ctx, cudaMemcpyAsync(seq_dev, seq_host, (size_t)n, cudaMemcpyHostToDevice, st));
    rc = rna4r_fold(ctx, seq_dev, n, score_dev, table_dev, table_dtype, workspace_dev, core, st);
    if (rc != RNA4R_OK) return rc;
    const int launches = ctx->last_launches;
    RNA4R_CUDA(ctx, cudaMemcpyAsync(score_out_host, score_dev, 4, cudaMemcpyDeviceToHost, st));
    if (table_bytes) RNA4R_CUDA(ctx, cudaMemcpyAsync(table_out_host, table_dev, table_bytes, cudaMemcpyDeviceToHost, st));
    RNA4R_CUDA(ctx, cudaStreamSynchronize(st));
    ctx->last_launches = launches;
    return RNA4R_OK;
}

int rna4r_fold_batch_host(rna4r_ctx *ctx, const uint8_t *seqs_host, const int32_t *lens_host, int count,
                          int32_t *scores_out_host, void *workspace_dev, size_t workspace_bytes, void *stream)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (count < 0) return RNA4R_ERR_BAD_N;
    if (count == 0) return RNA4R_OK;
    if (!lens_host || !scores_out_host || !workspace_dev) return RNA4R_ERR_NULL;
    size_t total_bases = 0;
    for (int t = 0; t < count; ++t) {
        int rc = check_n(ctx, lens_host[t]);
        if (rc != RNA4R_OK) return rc;
        total_bases += (size_t)lens_host[t];
    }
    if (!seqs_host && total_bases > 0) return RNA4R_ERR_NULL;
    if (workspace_bytes < rna4r_workspace_bytes_host(ctx, lens_host, count, RNA4R_TABLE_NONE)) return RNA4R_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    RNA4R_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t core = align_up(engine_ws(ctx, lens_host, count, 0), 256);
    char *stg = (char *)workspace_dev + core;
    uint8_t *seqs_dev = (uint8_t *)stg; stg += align_up(total_bases + 16, 256);
    int64_t *offs_dev = (int64_t *)stg; stg += align_up((size_t)(count + 1) * 8, 256);
    int32_t *scores_dev = (int32_t *)stg;
    // The offsets are an exclusive scan of the lengths, done on the device: the lengths travel in the (still unused)
    // score slots, so the call needs no host scratch and synchronises once, at the end.
    RNA4R_CUDA(ctx, cudaMemcpyAsync(scores_dev, lens_host, (size_t)count * 4, cudaMemcpyHostToDevice, st));
    if (total_bases) RNA4R_CUDA(ctx, cudaMemcpyAsync(seqs_dev, seqs_host, total_bases, cudaMemcpyHostToDevice, st));
    rna4r_offsets_from_lens_kernel<<<1, 1024, 0, st>>>(scores_dev, count, offs_dev);
    int rc = rna4r_fold_batch(ctx, seqs_dev, offs_dev, lens_host, count, scores_dev, workspace_dev, core, st);
    if (rc != RNA4R_OK) return rc;
    const int launches = ctx->last_launches + 1;
    RNA4R_CUDA(ctx, cudaMemcpyAsync(scores_out_host, scores_dev, (size_t)count * 4, cudaMemcpyDeviceToHost, st));
    RNA4R_CUDA(ctx, cudaStreamSynchronize(st));
    ctx->last_launches = launches;
    return RNA4R_OK;
}


// ---- rna4r_fold_static: a fold that allocates nothing and takes no workspace (include/rna4r.h) ------------------------
// The scratch of the tiled engine (plan, flags, super-tile records, bulk maxima) lives in this file-scope device array:
// RNA4R_STATIC_SCRATCH_BYTES on every GPU that loads the library, until the process exits.  In host code the NAME of the
// array is a host-side stand-in, not a device address: the address the kernels get is asked for once per device with
// cudaGetSymbolAddress (rna4r_fold_static_setup) and kept in g_static_scratch[device].
static __device__ __align__(256) unsigned char rna4r_static_scratch[RNA4R_STATIC_SCRATCH_BYTES];

namespace {
constexpr int kStaticMaxDevices = 64;
constexpr size_t kStaticTail = 512;                  // end of the array: the warm-up fold's sequence (256 B) and score
void *g_static_scratch[kStaticMaxDevices] = {nullptr};

inline size_t static_ws_limit() { return (size_t)RNA4R_STATIC_SCRATCH_BYTES - kStaticTail; }

int static_enqueue(rna4r_ctx *ctx, void *scratch, const uint8_t *seq_dev, int n, int32_t *score_dev, cudaStream_t st)
{
    // the tiled engine zeroes the prefix of its workspace that has to start at zero (plan header, flags) in every fold
    return dispatch_q(ctx->q, [&](auto Q) {
        return tiled::enqueue_q<decltype(Q)::value>(ctx, kDelta, seq_dev, nullptr, nullptr, 1, n, score_dev, nullptr, nullptr,
                                                    RNA4R_TABLE_NONE, scratch, st);
    });
}
}  // namespace

int rna4r_fold_static_max_n(const rna4r_ctx *ctx)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (ctx->q > 11) return RNA4R_ERR_ENGINE;
    int lo = 0, hi = 65534;                          // the workspace grows with n
    while (lo < hi) {
        const int mid = (lo + hi + 1) / 2;
        if (tiled_ws(ctx, nullptr, 1, mid) <= static_ws_limit()) lo = mid; else hi = mid - 1;
    }
    return lo;
}

int rna4r_fold_static_setup(rna4r_ctx *ctx, void *stream)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (ctx->q > 11) return RNA4R_ERR_ENGINE;
    if (ctx->device < 0 || ctx->device >= kStaticMaxDevices) return RNA4R_ERR_DEVICE;
    cudaStream_t st = (cudaStream_t)stream;
    RNA4R_CUDA(ctx, cudaSetDevice(ctx->device));
    void *ptr = nullptr;
    RNA4R_CUDA(ctx, cudaGetSymbolAddress(&ptr, rna4r_static_scratch));
    if (!ptr) return RNA4R_ERR_CUDA;
    // warm-up fold of 100 x 'A' out of the array's tail: module loading, kernel attributes and the occupancy query of
    // this context's q happen here, not in the first rna4r_fold_static call
    unsigned char *tailp = (unsigned char *)ptr + static_ws_limit();
    RNA4R_CUDA(ctx, cudaMemsetAsync(tailp, 'A', 256, st));
    int rc = static_enqueue(ctx, ptr, tailp, 100, (int32_t *)(tailp + 256), st);
    if (rc != RNA4R_OK) return rc;
    RNA4R_CUDA(ctx, cudaStreamSynchronize(st));
    g_static_scratch[ctx->device] = ptr;
    return RNA4R_OK;
}

int rna4r_fold_static(rna4r_ctx *ctx, const uint8_t *seq_dev, int n, int32_t *score_out_dev, void *stream)
{
    if (!ctx_ok(ctx)) return RNA4R_ERR_CONTEXT;
    if (ctx->q > 11) return RNA4R_ERR_ENGINE;
    if (!score_out_dev || (!seq_dev && n > 0)) return RNA4R_ERR_NULL;
    if (n < 0 || n > 65534) return RNA4R_ERR_BAD_N;
    if (tiled_ws(ctx, nullptr, 1, n) > static_ws_limit()) return RNA4R_ERR_BAD_N;       // beyond rna4r_fold_static_max_n
    if (ctx->device < 0 || ctx->device >= kStaticMaxDevices) return RNA4R_ERR_DEVICE;
    void *scratch = g_static_scratch[ctx->device];
    if (!scratch) return RNA4R_ERR_SETUP;
    RNA4R_CUDA(ctx, cudaSetDevice(ctx->device));
    return static_enqueue(ctx, scratch, seq_dev, n, score_out_dev, (cudaStream_t)stream);
}

}  // extern "C"
