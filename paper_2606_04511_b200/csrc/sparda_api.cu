// libsparda: context, argument validation and the Algorithm-2 stream choreography (include/sparda.h).
#include <alloca.h>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "sparda_internal.cuh"

int sparda_set_cuda_error(sparda_ctx* ctx, cudaError_t e, const char* where) {
    if (ctx) snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "%s: %s (%s)", cudaGetErrorName(e), cudaGetErrorString(e), where);
    (void)cudaGetLastError();
    return SPARDA_ECUDA;
}

extern "C" {

const char* sparda_version(void) { return "libsparda 0.1 (sm_100a)"; }

const char* sparda_strerror(int code) {
    switch (code) {
        case SPARDA_OK: return "ok";
        case SPARDA_EINVAL: return "invalid argument (null or misaligned pointer, or shape outside the supported set)";
        case SPARDA_EUNSUPPORTED: return "unsupported device (libsparda needs an sm_100 GPU)";
        case SPARDA_ECUDA: return "CUDA call failed (see sparda_last_cuda_error)";
        case SPARDA_ENOMEM: return "workspace allocation failed";
        case SPARDA_ELIMIT: return "shape beyond the fixed capacity of the no-allocation entry point (see sparda_noalloc_last_error)";
        default: return "unknown error code";
    }
}

const char* sparda_last_cuda_error(const sparda_ctx* ctx) { return ctx ? ctx->cuda_err : ""; }
int64_t sparda_launch_count(const sparda_ctx* ctx) { return ctx ? ctx->launches : 0; }
int64_t sparda_tmap_encodes(const sparda_ctx* ctx) { return ctx ? ctx->tmap_encodes : 0; }
int sparda_get_select_cluster(const sparda_ctx* ctx) { return ctx ? ctx->last_select_cluster : SPARDA_EINVAL; }
int sparda_get_attn_cluster(const sparda_ctx* ctx) { return ctx ? ctx->last_attn_cluster : SPARDA_EINVAL; }
int sparda_get_attn_splits(const sparda_ctx* ctx, int topk) { return ctx ? sparda_resolve_splits(ctx, topk) : SPARDA_EINVAL; }
int sparda_get_gather_ctas(const sparda_ctx* ctx) { return ctx ? ctx->cfg.gather_ctas : SPARDA_EINVAL; }

int sparda_create(const sparda_config* cfg, sparda_ctx** out) {
    if (!cfg || !out) return SPARDA_EINVAL;
    const int G = cfg->n_kv_heads > 0 ? cfg->n_q_heads / cfg->n_kv_heads : 0;
    if (cfg->batch < 1 || cfg->n_kv_heads < 1 || cfg->n_q_heads < 1 || cfg->n_q_heads % cfg->n_kv_heads != 0) return SPARDA_EINVAL;
    if (!(G == 1 || G == 2 || G == 4 || G == 8 || G == 16)) return SPARDA_EINVAL;
    if (cfg->head_dim != 64 && cfg->head_dim != 128) return SPARDA_EINVAL;
    if (cfg->block_size != 64) return SPARDA_EINVAL;
    if (cfg->max_blocks < 1 || cfg->max_blocks > 8192) return SPARDA_EINVAL;
    if (cfg->topk < 1 || cfg->topk > 256) return SPARDA_EINVAL;
    if (cfg->gather_mode != SPARDA_GATHER_TMA && cfg->gather_mode != SPARDA_GATHER_LDG) return SPARDA_EINVAL;
    if (cfg->gather_ctas < 0 || cfg->gather_ctas > 1024 || cfg->attn_splits < 0 || cfg->max_layers < 0) return SPARDA_EINVAL;
    if (cfg->attn_impl != 0 && cfg->attn_impl != 1) return SPARDA_EINVAL;
    if (cfg->hidden != 0 && (cfg->hidden < 64 || cfg->hidden > 8192 || cfg->hidden % 64 != 0)) return SPARDA_EINVAL;
    if (!(cfg->select_cluster == 0 || cfg->select_cluster == 1 || cfg->select_cluster == 2 || cfg->select_cluster == 4 ||
          cfg->select_cluster == 8 || cfg->select_cluster == 16))
        return SPARDA_EINVAL;

    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return SPARDA_EUNSUPPORTED;
    }
    if (prop.major != 10) return SPARDA_EUNSUPPORTED;

    sparda_ctx* ctx = new (std::nothrow) sparda_ctx();
    if (!ctx) return SPARDA_ENOMEM;
    memset(ctx, 0, sizeof(*ctx));
    ctx->cfg = *cfg;
    ctx->pdl_next = 1;
    ctx->device = dev;
    ctx->sm_count = prop.multiProcessorCount;
    ctx->R = cfg->batch * cfg->n_kv_heads;
    ctx->G = G;
    if (ctx->cfg.gather_ctas == 0) ctx->cfg.gather_ctas = cfg->gather_mode == SPARDA_GATHER_TMA ? 8 : 16;
    ctx->max_layers = cfg->max_layers > 0 ? cfg->max_layers : 64;
    {   // partial slots per row of the flat split-K attention: n_parts <= ceil(CTAs / R) + 1
        int per_row = cfg->attn_splits > 0 ? cfg->attn_splits : (2 * ctx->sm_count + ctx->R - 1) / ctx->R;
        if (per_row > cfg->topk) per_row = cfg->topk;
        ctx->max_splits = per_row + 2;
    }

    cudaError_t e;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
        (void)cudaGetLastError();
        delete ctx;
        return SPARDA_EUNSUPPORTED;
    }
    ctx->encode_fn = fn;

    const size_t D = cfg->head_dim;
    size_t n_po = (size_t)ctx->R * ctx->max_splits * SPARDA_MAX_G * D;
    size_t n_ml = (size_t)ctx->R * ctx->max_splits * 2 * SPARDA_MAX_G;
    bool ok = cudaMalloc(&ctx->part_O, n_po * sizeof(float)) == cudaSuccess &&
              cudaMalloc(&ctx->part_ml, n_ml * sizeof(float)) == cudaSuccess &&
              cudaMalloc(&ctx->tickets, (size_t)ctx->R * sizeof(unsigned int)) == cudaSuccess &&
              cudaMalloc(&ctx->probe_sink, 256 * sizeof(uint32_t)) == cudaSuccess &&
              cudaMalloc(&ctx->door, (size_t)(ctx->max_layers + 1) * sizeof(unsigned int)) == cudaSuccess &&
              cudaMemset(ctx->door, 0, (size_t)(ctx->max_layers + 1) * sizeof(unsigned int)) == cudaSuccess &&
              cudaMalloc(&ctx->pf_scratch, (size_t)ctx->sm_count * 512 * 128 * sizeof(float)) == cudaSuccess &&
              cudaMemset(ctx->tickets, 0, (size_t)ctx->R * sizeof(unsigned int)) == cudaSuccess;
    int prio_lo = 0, prio_hi = 0;
    ctx->ev_sel = (cudaEvent_t*)calloc(ctx->max_layers + 1, sizeof(cudaEvent_t));
    ctx->ev_gather = (cudaEvent_t*)calloc(ctx->max_layers + 1, sizeof(cudaEvent_t));
    ctx->ev_top = (cudaEvent_t*)calloc(ctx->max_layers + 1, sizeof(cudaEvent_t));
    ctx->ev_prof = (cudaEvent_t*)calloc((size_t)3 * (ctx->max_layers + 1) * 2, sizeof(cudaEvent_t));
    ok = ok && ctx->ev_sel && ctx->ev_gather && ctx->ev_top && ctx->ev_prof &&
         cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi) == cudaSuccess &&
         // highest priority: beside a many-CTA kernel of the caller's (a layer's GEMVs) the block scheduler hands SM slots to
         // the pending CTAs of the older kernel first; at equal priority the select waits for most of that kernel
         // (measured: 42 us instead of 20 beside a 4736-CTA stream).  Give the prefetch stream the same.
         cudaStreamCreateWithPriority(&ctx->select_stream, cudaStreamNonBlocking, prio_hi) == cudaSuccess;
    for (int i = 0; ok && i <= ctx->max_layers; ++i)
        ok = cudaEventCreateWithFlags(&ctx->ev_sel[i], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&ctx->ev_gather[i], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&ctx->ev_top[i], cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; ok && i < 3 * (ctx->max_layers + 1) * 2; ++i) ok = cudaEventCreate(&ctx->ev_prof[i]) == cudaSuccess;
    const size_t f_bytes = (size_t)ctx->R * D * 2, q_bytes = (size_t)cfg->batch * cfg->n_q_heads * D * 2;
    ok = ok && cudaMalloc(&ctx->stage_F, f_bytes * (ctx->max_layers + 1)) == cudaSuccess &&
         cudaMalloc(&ctx->stage_Q, q_bytes * ctx->max_layers) == cudaSuccess &&
         cudaMalloc(&ctx->stage_O, q_bytes * ctx->max_layers) == cudaSuccess;
    if (!ok) {
        (void)cudaGetLastError();
        sparda_destroy(ctx);
        return SPARDA_ENOMEM;
    }
    if (cudaDeviceSynchronize() != cudaSuccess) {
        (void)cudaGetLastError();
        sparda_destroy(ctx);
        return SPARDA_ECUDA;
    }
    *out = ctx;
    return SPARDA_OK;
}

int sparda_destroy(sparda_ctx* ctx) {
    if (!ctx) return SPARDA_EINVAL;
    (void)cudaDeviceSynchronize();
    cudaFree(ctx->part_O);
    cudaFree(ctx->part_ml);
    cudaFree(ctx->tickets);
    cudaFree(ctx->pf_scratch);
    cudaFree(ctx->probe_sink);
    cudaFree(ctx->door);
    for (int i = 0; i <= ctx->max_layers; ++i) {
        if (ctx->ev_sel && ctx->ev_sel[i]) cudaEventDestroy(ctx->ev_sel[i]);
        if (ctx->ev_gather && ctx->ev_gather[i]) cudaEventDestroy(ctx->ev_gather[i]);
        if (ctx->ev_top && ctx->ev_top[i]) cudaEventDestroy(ctx->ev_top[i]);
    }
    for (int i = 0; ctx->ev_prof && i < 3 * (ctx->max_layers + 1) * 2; ++i)
        if (ctx->ev_prof[i]) cudaEventDestroy(ctx->ev_prof[i]);
    cudaFree(ctx->stage_F);
    cudaFree(ctx->stage_Q);
    cudaFree(ctx->stage_O);
    free(ctx->ev_sel);
    free(ctx->ev_gather);
    free(ctx->ev_top);
    if (ctx->select_stream) cudaStreamDestroy(ctx->select_stream);
    free(ctx->ev_prof);
    (void)cudaGetLastError();
    delete ctx;
    return SPARDA_OK;
}

int sparda_pool_keys(sparda_ctx* ctx, const void* kv, int64_t n_rows, int n_blocks, void* kpool, void* stream) {
    if (!ctx || !sparda_aligned(kv, 16) || !sparda_aligned(kpool, 16) || n_rows < 1 || n_blocks < 1) return SPARDA_EINVAL;
    if (n_rows * (int64_t)n_blocks > (int64_t)1 << 31) return SPARDA_EINVAL;
    return sparda_launch_pool_keys(ctx, kv, n_rows, n_blocks, kpool, (cudaStream_t)stream);
}

int sparda_forecast_project(sparda_ctx* ctx, const void* X, const void* WF, int hidden, void* F_out, void* stream) {
    if (!ctx || !sparda_aligned(X, 16) || !sparda_aligned(WF, 16) || !sparda_aligned(F_out, 16)) return SPARDA_EINVAL;
    if (hidden < 64 || hidden > 8192 || hidden % 64 != 0) return SPARDA_EINVAL;
    return sparda_launch_forecast_project(ctx, X, WF, hidden, F_out, (cudaStream_t)stream);
}

int sparda_append_kv(sparda_ctx* ctx, const void* k_new, const void* v_new, int64_t t, void* kv_cache, int n_blocks, float* ksum,
                     void* kpool, void* stream) {
    if (!ctx || !sparda_aligned(k_new, 16) || !sparda_aligned(v_new, 16) || !sparda_aligned(kv_cache, 16) || !sparda_aligned(ksum, 16) ||
        !sparda_aligned(kpool, 16))
        return SPARDA_EINVAL;
    if (n_blocks < 1 || n_blocks > ctx->cfg.max_blocks || t < 0 || t >= (int64_t)n_blocks * ctx->cfg.block_size) return SPARDA_EINVAL;
    return sparda_launch_append_kv(ctx, k_new, v_new, t, kv_cache, n_blocks, ksum, kpool, (cudaStream_t)stream);
}

int sparda_forecast_select(sparda_ctx* ctx, const void* F, const void* Kpool, int n_blocks, int n_cand, int topk,
                           int32_t* ids_out, void* stream) {
    if (!ctx || !sparda_aligned(F, 16) || !sparda_aligned(Kpool, 16) || !sparda_aligned(ids_out, 4)) return SPARDA_EINVAL;
    if (n_blocks < 1 || n_blocks > ctx->cfg.max_blocks || n_cand < 0 || n_cand > n_blocks) return SPARDA_EINVAL;
    if (topk < 1 || topk > ctx->cfg.topk) return SPARDA_EINVAL;
    return sparda_launch_select(ctx, F, Kpool, n_blocks, n_cand, topk, ids_out, nullptr, nullptr, nullptr, (cudaStream_t)stream);
}

int sparda_pool_keys_grid(sparda_ctx* ctx, const void* kv, int64_t n_rows, int n_blocks, void* kgrid, void* stream) {
    if (!ctx || !sparda_aligned(kv, 16) || !sparda_aligned(kgrid, 16) || n_rows < 1 || n_blocks < 1) return SPARDA_EINVAL;
    if (n_rows * (int64_t)n_blocks > (int64_t)1 << 29) return SPARDA_EINVAL;
    return sparda_launch_pool_keys_grid(ctx, kv, n_rows, n_blocks, kgrid, (cudaStream_t)stream);
}

int sparda_forecast_select_grid(sparda_ctx* ctx, const void* F, const void* Kgrid, int n_blocks, int n_cand, int n_init, int n_local,
                                int topk, int32_t* ids_out, void* stream) {
    if (!ctx || !sparda_aligned(F, 16) || !sparda_aligned(Kgrid, 16) || !sparda_aligned(ids_out, 4)) return SPARDA_EINVAL;
    if (n_blocks < 1 || n_blocks > ctx->cfg.max_blocks || n_cand < 0 || n_cand > n_blocks) return SPARDA_EINVAL;
    if (topk < 1 || topk > ctx->cfg.topk || n_init < 0 || n_local < 0 || n_init + n_local > topk) return SPARDA_EINVAL;
    return sparda_launch_select_grid(ctx, F, Kgrid, n_blocks, n_cand, n_init, n_local, topk, ids_out, (cudaStream_t)stream);
}

int sparda_forecast_select_plan(sparda_ctx* ctx, const void* F, const void* Kpool, int n_blocks, int n_cand, int topk,
                                int32_t* ids_out, int32_t* slot_ids, int32_t* fetch, int32_t* n_fetch, void* stream) {
    if (!ctx || !sparda_aligned(F, 16) || !sparda_aligned(Kpool, 16) || !sparda_aligned(ids_out, 4)) return SPARDA_EINVAL;
    if (!sparda_aligned(slot_ids, 4) || !sparda_aligned(fetch, 4) || (n_fetch && !sparda_aligned(n_fetch, 4))) return SPARDA_EINVAL;
    if (n_blocks < 1 || n_blocks > ctx->cfg.max_blocks || n_cand < 0 || n_cand > n_blocks) return SPARDA_EINVAL;
    if (topk < 1 || topk > ctx->cfg.topk) return SPARDA_EINVAL;
    return sparda_launch_select(ctx, F, Kpool, n_blocks, n_cand, topk, ids_out, slot_ids, fetch, n_fetch, (cudaStream_t)stream);
}

int sparda_prefetch_launch(sparda_ctx* ctx, const void* host_kv, int n_blocks, const int32_t* ids, int topk,
                           void* dev_pool, void* stream) {
    if (!ctx || !sparda_aligned(host_kv, 16) || !sparda_aligned(dev_pool, 16) || !sparda_aligned(ids, 4)) return SPARDA_EINVAL;
    if (n_blocks < 1 || n_blocks > ctx->cfg.max_blocks || topk < 1 || topk > ctx->cfg.topk) return SPARDA_EINVAL;
    return sparda_launch_gather(ctx, host_kv, n_blocks, ids, topk, dev_pool, (cudaStream_t)stream);
}

int sparda_enable_peer_tier(sparda_ctx* ctx, int peer_device) {
    if (!ctx) return SPARDA_EINVAL;
    int n = 0, can = 0, cur = -1;
    if (cudaGetDeviceCount(&n) != cudaSuccess) return sparda_set_cuda_error(ctx, cudaGetLastError(), "cudaGetDeviceCount");
    if (peer_device < 0 || peer_device >= n || peer_device == ctx->device) return SPARDA_EINVAL;
    SPARDA_CUDA_TRY(ctx, cudaDeviceCanAccessPeer(&can, ctx->device, peer_device));
    if (!can) return SPARDA_EUNSUPPORTED;
    SPARDA_CUDA_TRY(ctx, cudaGetDevice(&cur));
    if (cur != ctx->device) SPARDA_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaError_t e = cudaDeviceEnablePeerAccess(peer_device, 0);
    if (cur != ctx->device) (void)cudaSetDevice(cur);
    if (e == cudaErrorPeerAccessAlreadyEnabled) { (void)cudaGetLastError(); e = cudaSuccess; }
    if (e != cudaSuccess) return sparda_set_cuda_error(ctx, e, "cudaDeviceEnablePeerAccess");
    return SPARDA_OK;
}

int sparda_sparse_decode(sparda_ctx* ctx, const void* Q, const void* dev_pool, const int32_t* ids, int topk,
                         int pool_is_indexed, int n_slots, void* O, void* stream) {
    if (!ctx || !sparda_aligned(Q, 16) || !sparda_aligned(dev_pool, 16) || !sparda_aligned(ids, 4) || !sparda_aligned(O, 16))
        return SPARDA_EINVAL;
    if (topk < 1 || topk > ctx->cfg.topk) return SPARDA_EINVAL;
    if (pool_is_indexed ? (n_slots < 1 || n_slots > ctx->cfg.max_blocks) : (n_slots != topk)) return SPARDA_EINVAL;
    return sparda_launch_attn(ctx, Q, dev_pool, ids, nullptr, topk, pool_is_indexed ? 1 : 0, n_slots, O, (cudaStream_t)stream);
}

int sparda_sparse_decode_varlen(sparda_ctx* ctx, const void* Q, const void* dev_pool, const int32_t* ids, const int32_t* seq_len, int topk,
                                int pool_is_indexed, int n_slots, void* O, void* stream) {
    if (!ctx || !sparda_aligned(Q, 16) || !sparda_aligned(dev_pool, 16) || !sparda_aligned(ids, 4) || !sparda_aligned(O, 16) ||
        !sparda_aligned(seq_len, 4))
        return SPARDA_EINVAL;
    if (topk < 1 || topk > ctx->cfg.topk) return SPARDA_EINVAL;
    if (pool_is_indexed ? (n_slots < 1 || n_slots > ctx->cfg.max_blocks) : (n_slots != topk)) return SPARDA_EINVAL;
    return sparda_launch_attn(ctx, Q, dev_pool, ids, seq_len, topk, pool_is_indexed ? 1 : 0, n_slots, O, (cudaStream_t)stream);
}

int sparda_prefill_select(sparda_ctx* ctx, const void* F, const void* Kpool, int T, int n_blocks, int row0, int n_rows,
                          int topk, int32_t* ids_out, void* stream) {
    if (!ctx || !sparda_aligned(F, 16) || !sparda_aligned(Kpool, 16) || !sparda_aligned(ids_out, 16)) return SPARDA_EINVAL;
    if (T < 1 || n_blocks < 1 || n_blocks > ctx->cfg.max_blocks || row0 < 0 || n_rows < 1 || row0 + (int64_t)n_rows > T) return SPARDA_EINVAL;
    if (topk < 1 || topk > ctx->cfg.topk) return SPARDA_EINVAL;
    return sparda_launch_prefill_select(ctx, F, Kpool, T, n_blocks, row0, n_rows, topk, ids_out, (cudaStream_t)stream);
}

int sparda_prefill_select_baseline(sparda_ctx* ctx, const void* Q, const void* Kpool, int T, int n_blocks, int row0,
                                   int n_rows, int topk, int32_t* ids_out, void* stream) {
    if (!ctx || !sparda_aligned(Q, 16) || !sparda_aligned(Kpool, 16) || !sparda_aligned(ids_out, 16)) return SPARDA_EINVAL;
    if (T < 1 || n_blocks < 1 || n_blocks > ctx->cfg.max_blocks || row0 < 0 || n_rows < 1 || row0 + (int64_t)n_rows > T) return SPARDA_EINVAL;
    if (topk < 1 || topk > ctx->cfg.topk) return SPARDA_EINVAL;
    return sparda_launch_prefill_baseline(ctx, Q, Kpool, T, n_blocks, row0, n_rows, topk, ids_out, (cudaStream_t)stream);
}

// Algorithm 2, lines 4-7, for n_layers layers, plain (double-buffered pool, every block fetched) or with the
// previous step's blocks kept per layer.  Given layer l's projections, line 4 (select B_{l+1}) and line 7
// (attention l) do not depend on each other, so in overlap mode they run concurrently on two streams; the prefetch has
// its own, on which the gathers run one after the other, each alone on the link:
//   compute stream  cs:  record ev_top[l]  ->  wait ev_gather[l] (and ev_sel[l])  ->  attention l
//   select stream   ss:  wait ev_top[l]    ->  [F_l = X_l W_F]  ->  select B_{l+1} (+ reuse plan), rings door[l+1] row by row  ->  record ev_sel[l+1]
//   prefetch stream ps:  wait ev_top[l]    ->  gather B_{l+1}: waits ON THE DEVICE for door[l+1] == R, copies  ->  record ev_gather[l+1]
// ev_top[l] follows attention l-1 on cs, so a select never runs more than one layer ahead of the attention (in a model,
// F_l exists only once layer l-1 is complete) and it releases the buffers gather l+1 writes: pool[(l+1)&1] was last read
// by attention l-1 (plain); pool_{l+1} and slot_ids_{l+1} by attention l+1 of the previous step (cached).
// The doorbell (sparda_internal.cuh) takes the select -> gather kernel boundary off the chain: the gather launch is resident
// (8 one-warp CTAs, sleeping between polls) while the select runs and starts the moment the last row's list is out.  Alone the
// boundary costs ~3 us; beside a kernel that saturates the GPU -- a real layer -- a dependent launch costs 10-20 us and the chain
// select -> gather 40 us instead of 9 (measured), which is what bounds how much link time fits behind a layer.
// Every gather ends in an event an attention waits for, and ev_sel joins the select stream, so cs has joined both side
// streams when the step ends (capturable).  A cross-stream hand-off costs next to nothing inside a CUDA graph when the GPU
// is idle (measured); putting a layer's select and gather on one stream and alternating two such streams between layers was
// tried: same floor, but two gathers then share the link and the step with every block fetched loses 1 %.  Serial mode: the
// same kernels on cs in Algorithm-2 order, no doorbell.
// timing events around one launch of `kind` (0 select, 1 gather, 2 attention) on stream st
static inline cudaEvent_t* prof_slot(sparda_ctx* ctx, int kind) {
    return &ctx->ev_prof[((size_t)kind * (ctx->max_layers + 1) + ctx->prof_n[kind]) * 2];
}
#define SPARDA_PROF_BEGIN(kind, st) \
    if (ctx->prof_on) SPARDA_CUDA_TRY(ctx, cudaEventRecord(prof_slot(ctx, kind)[0], st))
#define SPARDA_PROF_END(kind, st)                                               \
    if (ctx->prof_on) {                                                         \
        SPARDA_CUDA_TRY(ctx, cudaEventRecord(prof_slot(ctx, kind)[1], st));     \
        ctx->prof_n[kind]++;                                                    \
    }

// Host-buffer form (sparda_decode_step_host): the caller's F / Q / O live in pinned host memory.  Their copies are
// enqueued on the compute stream just in time -- F_l and Q_l before layer l begins, O_l right after attention l -- so
// they run while that stream waits for a gather instead of in front of and behind the whole step.
struct HostIO {
    const sparda_layer* host;   // host pointers F, Q, O per layer
    const void* F0cur;          // host
    size_t f_bytes, q_bytes;
};

static int decode_step_impl(sparda_ctx* ctx, const sparda_cached_layer* layers, int n_layers, const void* F0cur, int n_blocks,
                            int topk, cudaStream_t cs, cudaStream_t ps_in, int mode, const HostIO* io = nullptr) {
    const bool overlap = mode == SPARDA_STEP_OVERLAP;
    // candidate range of every selection of the step: the complete blocks of a cache of capacity n_blocks (sparda_set_step_candidates)
    const int n_cand = ctx->step_n_cand > 0 && ctx->step_n_cand < n_blocks ? ctx->step_n_cand : n_blocks;
    cudaStream_t ss = overlap ? ctx->select_stream : cs, ps = overlap ? ps_in : cs;
    int rc;
    ctx->prof_n[0] = ctx->prof_n[1] = ctx->prof_n[2] = 0;
    // doorbells of this step: every door of the previous step has been consumed (the compute stream joined both side streams)
    if (overlap) SPARDA_CUDA_TRY(ctx, cudaMemsetAsync(ctx->door, 0, (size_t)(n_layers + 1) * sizeof(unsigned int), cs));
    if (io) SPARDA_CUDA_TRY(ctx, cudaMemcpyAsync(const_cast<void*>(F0cur), io->F0cur, io->f_bytes, cudaMemcpyHostToDevice, cs));
    // layer 0: same-layer selection with F0cur; its attention needs it, so it stays on the compute stream
    if (!io && layers[0].base.X && layers[0].base.WFcur) {   // Alg.2 l.1 for F_0^cur (Eq.3)
        if (!ctx->cfg.hidden) return SPARDA_EINVAL;
        rc = sparda_launch_forecast_project(ctx, layers[0].base.X, layers[0].base.WFcur, ctx->cfg.hidden, const_cast<void*>(F0cur), cs);
        if (rc) return rc;
    }
    SPARDA_PROF_BEGIN(0, cs);
    // f3 inside the step (sparda_set_step_selector): Kpool then is the (32,16) compressed-key grid [R][4 n_blocks][D] and every
    // selection returns init + local + top-k (reading q19, unpinned by the paper)
    const bool grid = ctx->step_grid != 0;
    if (grid && ctx->step_n_init + ctx->step_n_local > topk) return SPARDA_EINVAL;
    rc = grid ? sparda_forecast_select_grid(ctx, F0cur, layers[0].base.Kpool, n_blocks, n_cand, ctx->step_n_init, ctx->step_n_local, topk,
                                            layers[0].base.ids, cs)
              : sparda_forecast_select(ctx, F0cur, layers[0].base.Kpool, n_blocks, n_cand, topk, layers[0].base.ids, cs);
    if (rc) return rc;
    SPARDA_PROF_END(0, cs);
    // Doorbell admission.  A waiting gather CTA holds its SM slot (TMA engine: ~104 KB of shared memory, two fit per SM; LDG
    // engine: 256 threads, eight fit) until the select has rung, and nothing orders "select resident before gather" on the
    // device -- least of all in a CUDA-graph replay, where the two are independent nodes.  With at most sm_count / 2 gather CTAs
    // at least half of the SMs hold no gather CTA whatever the placement, so the select's clusters (and the attention) can
    // always be scheduled and the wait ends.  Beyond that (cfg.gather_ctas up to 1024 is accepted, the peer tier asks for more
    // CTAs) a grid of spinning CTAs could occupy every SM and the step would trap after ~15 s: such a grid is not given a door.
    const bool door_fits = 2 * ctx->cfg.gather_ctas <= ctx->sm_count;
    struct PdlScope {   // launches behind an event wait do not ask for PDL (see sparda_ctx::pdl_next); restored on every return
        sparda_ctx* c;
        ~PdlScope() { c->pdl_next = 1; }
    } pdl_scope{ctx};
    for (int l = 0; l < n_layers; ++l) {
        if (io) {   // this layer's Forecast and query, before ev_top[l] releases the select that reads F_l
            if (l + 1 < n_layers)
                SPARDA_CUDA_TRY(ctx, cudaMemcpyAsync(const_cast<void*>(layers[l].base.F), io->host[l].F, io->f_bytes, cudaMemcpyHostToDevice, cs));
            SPARDA_CUDA_TRY(ctx, cudaMemcpyAsync(const_cast<void*>(layers[l].base.Q), io->host[l].Q, io->q_bytes, cudaMemcpyHostToDevice, cs));
        }
        if (l + 1 < n_layers) {
            const sparda_cached_layer* nx = &layers[l + 1];
            cudaStream_t xs = ss, gs = ps;
            if (overlap) {
                SPARDA_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_top[l], cs));
                SPARDA_CUDA_TRY(ctx, cudaStreamWaitEvent(xs, ctx->ev_top[l], 0));
            }
            ctx->pdl_next = overlap ? 0 : 1;   // overlap mode launches without PDL (measured: 0.38 ms per cached step against 0.43)
            if (!io && layers[l].base.X && layers[l].base.WF) {   // Alg.2 l.1: F_l = X_l . W_F (Eq.3), where its reader runs
                if (!ctx->cfg.hidden) return SPARDA_EINVAL;
                rc = sparda_launch_forecast_project(ctx, layers[l].base.X, layers[l].base.WF, ctx->cfg.hidden, const_cast<void*>(layers[l].base.F), xs);
                if (rc) return rc;
                ctx->pdl_next = 1;   // the select follows the projection on its own stream, no event in between: its prologue
                                     // and the first ring of pooled keys overlap the projection (0.58 -> 0.55 ms per cached step, batch 4)
            }
            // the doorbell needs the list the gather reads to come out of the ringing kernel: not so for grid select + separate plan.
            // It also needs the select to become resident while the gather CTAs spin: guaranteed only when the gather grid cannot
            // fill the device (door_fits below); a larger grid is ordered behind the select by ev_sel, like grid + plan
            const bool use_door = overlap && door_fits && !(grid && nx->slot_ids);
            ctx->door_next = use_door ? ctx->door + (l + 1) : nullptr;   // this select rings the layer's gather (below) row by row
            SPARDA_PROF_BEGIN(0, xs);
            if (grid) {
                rc = sparda_forecast_select_grid(ctx, layers[l].base.F, nx->base.Kpool, n_blocks, n_cand, ctx->step_n_init, ctx->step_n_local,
                                                 topk, nx->base.ids, xs);
                if (!rc && nx->slot_ids) rc = sparda_reuse_plan(ctx, nx->base.ids, topk, nx->slot_ids, nx->fetch, nx->n_fetch, xs);
            } else if (nx->slot_ids)   // select + reuse plan in one launch
                rc = sparda_forecast_select_plan(ctx, layers[l].base.F, nx->base.Kpool, n_blocks, n_cand, topk, nx->base.ids,
                                                 nx->slot_ids, nx->fetch, nx->n_fetch, xs);
            else
                rc = sparda_forecast_select(ctx, layers[l].base.F, nx->base.Kpool, n_blocks, n_cand, topk, nx->base.ids, xs);
            if (rc) { ctx->door_next = nullptr; return rc; }
            SPARDA_PROF_END(0, xs);
            ctx->pdl_next = overlap ? 0 : 1;
            if (overlap) {
                // the gather does not wait for the select's kernel boundary: it starts with the select (both behind ev_top[l],
                // which also releases the pool it writes) and waits on the device for the doorbell.  ev_sel joins the select
                // stream back into the compute stream in front of attention l+1 (stream capture needs the join)
                SPARDA_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_sel[l + 1], xs));
                SPARDA_CUDA_TRY(ctx, cudaStreamWaitEvent(gs, use_door ? ctx->ev_top[l] : ctx->ev_sel[l + 1], 0));
            }
            SPARDA_PROF_BEGIN(1, gs);
            rc = sparda_prefetch_launch(ctx, nx->base.kv, n_blocks, nx->slot_ids ? nx->fetch : nx->base.ids, topk, nx->pool, gs);
            ctx->door_next = nullptr;
            if (rc) return rc;
            SPARDA_PROF_END(1, gs);
            if (overlap) SPARDA_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_gather[l + 1], gs));
        }
        ctx->pdl_next = overlap ? 0 : 1;       // the attention waits for its gather's event in overlap mode
        if (l == 0) {
            SPARDA_PROF_BEGIN(2, cs);
            rc = sparda_sparse_decode(ctx, layers[0].base.Q, layers[0].base.kv, layers[0].base.ids, topk, 1, n_blocks, layers[0].base.O, cs);
        } else {
            if (overlap) {
                SPARDA_CUDA_TRY(ctx, cudaStreamWaitEvent(cs, ctx->ev_gather[l], 0));
                SPARDA_CUDA_TRY(ctx, cudaStreamWaitEvent(cs, ctx->ev_sel[l], 0));
            }
            SPARDA_PROF_BEGIN(2, cs);
            rc = sparda_sparse_decode(ctx, layers[l].base.Q, layers[l].pool, layers[l].slot_ids ? layers[l].slot_ids : layers[l].base.ids,
                                      topk, 0, topk, layers[l].base.O, cs);
        }
        if (rc) return rc;
        SPARDA_PROF_END(2, cs);
        if (ctx->standin_buf) {   // measurement only: the rest of layer l (weights streamed once), between attention l and layer l+1
            rc = sparda_launch_standin(ctx, cs);
            if (rc) return rc;
        }
        if (io) SPARDA_CUDA_TRY(ctx, cudaMemcpyAsync(io->host[l].O, layers[l].base.O, io->q_bytes, cudaMemcpyDeviceToHost, cs));
    }
    // every chain ended in an ev_gather that an attention on cs waited for: cs has joined both side streams (capturable)
    return SPARDA_OK;
}

int sparda_decode_step(sparda_ctx* ctx, const sparda_layer* layers, int n_layers, const void* F0cur, int n_blocks,
                       int topk, void* dev_pool0, void* dev_pool1, void* compute_stream, void* prefetch_stream,
                       int mode) {
    if (!ctx || !layers || n_layers < 1 || n_layers > ctx->max_layers || !F0cur) return SPARDA_EINVAL;
    if (mode != SPARDA_STEP_OVERLAP && mode != SPARDA_STEP_SERIAL) return SPARDA_EINVAL;
    if (n_layers > 1 && (!dev_pool0 || !dev_pool1)) return SPARDA_EINVAL;
    void* pools[2] = {dev_pool0, dev_pool1};
    sparda_cached_layer* cl = (sparda_cached_layer*)alloca(sizeof(sparda_cached_layer) * (size_t)n_layers);
    for (int l = 0; l < n_layers; ++l) {
        cl[l].base = layers[l];
        cl[l].pool = pools[l & 1];   // double-buffered: gather l+1 lands while attention l reads the other buffer
        cl[l].slot_ids = nullptr;
        cl[l].fetch = nullptr;
        cl[l].n_fetch = nullptr;
    }
    return decode_step_impl(ctx, cl, n_layers, F0cur, n_blocks, topk, (cudaStream_t)compute_stream, (cudaStream_t)prefetch_stream, mode);
}

int sparda_reuse_plan(sparda_ctx* ctx, const int32_t* ids_new, int topk, int32_t* slot_ids, int32_t* fetch, int32_t* n_fetch,
                      void* stream) {
    if (!ctx || !sparda_aligned(ids_new, 4) || !sparda_aligned(slot_ids, 4) || !sparda_aligned(fetch, 4)) return SPARDA_EINVAL;
    if (n_fetch && !sparda_aligned(n_fetch, 4)) return SPARDA_EINVAL;
    if (topk < 1 || topk > ctx->cfg.topk) return SPARDA_EINVAL;
    return sparda_launch_reuse_plan(ctx, ids_new, topk, slot_ids, fetch, n_fetch, (cudaStream_t)stream);
}

int sparda_decode_step_cached(sparda_ctx* ctx, const sparda_cached_layer* layers, int n_layers, const void* F0cur, int n_blocks,
                              int topk, void* compute_stream, void* prefetch_stream, int mode) {
    if (!ctx || !layers || n_layers < 1 || n_layers > ctx->max_layers || !F0cur) return SPARDA_EINVAL;
    if (mode != SPARDA_STEP_OVERLAP && mode != SPARDA_STEP_SERIAL) return SPARDA_EINVAL;
    for (int l = 1; l < n_layers; ++l)
        if (!layers[l].pool || !layers[l].slot_ids || !layers[l].fetch) return SPARDA_EINVAL;
    return decode_step_impl(ctx, layers, n_layers, F0cur, n_blocks, topk, (cudaStream_t)compute_stream, (cudaStream_t)prefetch_stream, mode);
}

int sparda_decode_step_host(sparda_ctx* ctx, const sparda_layer* layers, int n_layers, const void* F0cur, int n_blocks,
                            int topk, void* dev_pool0, void* dev_pool1, void* compute_stream, void* prefetch_stream,
                            int mode) {
    if (!ctx || !layers || n_layers < 1 || n_layers > ctx->max_layers || !F0cur) return SPARDA_EINVAL;
    cudaStream_t cs = (cudaStream_t)compute_stream;
    const size_t f_bytes = (size_t)ctx->R * ctx->cfg.head_dim * 2;
    const size_t q_bytes = (size_t)ctx->cfg.batch * ctx->cfg.n_q_heads * ctx->cfg.head_dim * 2;
    if (mode != SPARDA_STEP_OVERLAP && mode != SPARDA_STEP_SERIAL) return SPARDA_EINVAL;
    if (n_layers > 1 && (!dev_pool0 || !dev_pool1)) return SPARDA_EINVAL;
    void* pools[2] = {dev_pool0, dev_pool1};
    sparda_cached_layer* cl = (sparda_cached_layer*)alloca(sizeof(sparda_cached_layer) * (size_t)n_layers);
    for (int l = 0; l < n_layers; ++l) {
        if (!layers[l].Q || !layers[l].O || (l + 1 < n_layers && !layers[l].F)) return SPARDA_EINVAL;
        cl[l].base = layers[l];
        cl[l].base.F = ctx->stage_F + f_bytes * l;
        cl[l].base.Q = ctx->stage_Q + q_bytes * l;
        cl[l].base.O = ctx->stage_O + q_bytes * l;
        cl[l].pool = pools[l & 1];
        cl[l].slot_ids = nullptr;
        cl[l].fetch = nullptr;
        cl[l].n_fetch = nullptr;
    }
    HostIO io = {layers, F0cur, f_bytes, q_bytes};
    return decode_step_impl(ctx, cl, n_layers, ctx->stage_F + f_bytes * ctx->max_layers, n_blocks, topk, cs, (cudaStream_t)prefetch_stream, mode,
                            &io);
}

int sparda_set_step_selector(sparda_ctx* ctx, int grid, int n_init, int n_local) {
    if (!ctx || n_init < 0 || n_local < 0 || (grid != 0 && grid != 1)) return SPARDA_EINVAL;
    if (grid && n_init + n_local > ctx->cfg.topk) return SPARDA_EINVAL;
    ctx->step_grid = grid;
    ctx->step_n_init = grid ? n_init : 0;
    ctx->step_n_local = grid ? n_local : 0;
    return SPARDA_OK;
}

int sparda_set_step_candidates(sparda_ctx* ctx, int n_cand) {
    if (!ctx || n_cand < 0) return SPARDA_EINVAL;
    ctx->step_n_cand = n_cand;
    return SPARDA_OK;
}

int sparda_profile_enable(sparda_ctx* ctx, int on) {
    if (!ctx) return SPARDA_EINVAL;
    ctx->prof_on = on ? 1 : 0;
    ctx->prof_n[0] = ctx->prof_n[1] = ctx->prof_n[2] = 0;
    return SPARDA_OK;
}

int sparda_profile_read(sparda_ctx* ctx, double ms_out[3], int64_t count_out[3]) {
    if (!ctx || !ms_out || !count_out) return SPARDA_EINVAL;
    for (int k = 0; k < 3; ++k) {
        double sum = 0.0;
        for (int i = 0; i < ctx->prof_n[k]; ++i) {
            cudaEvent_t* e = &ctx->ev_prof[((size_t)k * (ctx->max_layers + 1) + i) * 2];
            float ms = 0.f;
            SPARDA_CUDA_TRY(ctx, cudaEventSynchronize(e[1]));
            SPARDA_CUDA_TRY(ctx, cudaEventElapsedTime(&ms, e[0], e[1]));
            sum += ms;
        }
        ms_out[k] = sum;
        count_out[k] = ctx->prof_n[k];
    }
    return SPARDA_OK;
}

}  // extern "C"

// TMA descriptor for a [rows][head_dim] bf16 view (KV pool / cache, F, Kpool): box = box_rows x 64 elements (128 B),
// 128-byte swizzle.  Cached per (base, rows, head_dim, box_rows) in an open-addressed hash table: encoding costs a few
// microseconds on the host.  The caller receives a copy (kernels take it as a __grid_constant__ parameter), so a later
// lookup that evicts an entry cannot change a descriptor already handed out.
int sparda_get_tmap(sparda_ctx* ctx, const void* base, uint64_t rows, int head_dim, int box_rows, CUtensorMap* out) {
    uint64_t h = (uint64_t)(uintptr_t)base * 0x9E3779B97F4A7C15ull ^ rows * 0xC2B2AE3D27D4EB4Full ^ (uint64_t)(head_dim * 131 + box_rows);
    h ^= h >> 29;
    const int home = (int)(h & (SPARDA_TMAP_SLOTS - 1));
    sparda_tmap_entry* e = nullptr;
    for (int probe = 0; probe < 8; ++probe) {
        sparda_tmap_entry* c = &ctx->tmaps[(home + probe) & (SPARDA_TMAP_SLOTS - 1)];
        if (c->base == base && c->rows == rows && c->head_dim == head_dim && c->box_rows == box_rows) {
            *out = c->map;
            return SPARDA_OK;
        }
        if (!c->base) { e = c; break; }
    }
    if (!e) e = &ctx->tmaps[home];   // neighbourhood full: overwrite the home slot
    typedef CUresult (*encode_t)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    cuuint64_t gdim[2] = {(cuuint64_t)head_dim, (cuuint64_t)rows};
    cuuint64_t gstride[1] = {(cuuint64_t)head_dim * 2};
    cuuint32_t box[2] = {64, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = ((encode_t)ctx->encode_fn)(&e->map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), gdim, gstride, box,
                                            estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
        e->base = nullptr;
        return SPARDA_ECUDA;
    }
    e->base = base;
    e->rows = rows;
    e->head_dim = head_dim;
    e->box_rows = box_rows;
    ctx->tmap_encodes++;
    *out = e->map;
    return SPARDA_OK;
}
