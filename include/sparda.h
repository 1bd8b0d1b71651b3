/*
 * sparda.h -- C ABI of libsparda: SparDA's decode-time hot path, hand-written CUDA for sm_100a (B200).
 *
 * Citations: P:L<n> = line n of the paper text (arxiv 2606.04511, "SparDA: Sparse Decoupled Attention
 * for Efficient Long-Context LLM Inference"); section / equation / algorithm named beside it.
 *
 * The path (Algorithm 2, lines 4-7), per layer l of one decode step:
 *   4  B_{l+1} <- f_top(F_l Kpool_{l+1}^T, k)      sparda_forecast_select      (Eq.4)
 *   5  launch prefetch of B_{l+1}, CPU -> GPU       sparda_prefetch_launch      (Sec.4.3)
 *   6  wait for the KV entries of B_l               events, sparda_decode_step
 *   7  O_l <- Attn(Q_l, K_l[B_l], V_l[B_l])         sparda_sparse_decode        (Eq.5)
 * plus the selection line of the prefill step (Algorithm 1 line 2): sparda_prefill_select and the
 * multi-head softmax selector it replaces: sparda_prefill_select_baseline.
 *
 * Conventions
 *  - Plain C linkage, plain pointers and sizes.  "device" = pointer valid in device code on the current
 *    CUDA device; "host-mapped" = device-visible pointer to pinned (page-locked, mapped) host memory
 *    (cudaHostAlloc / cudaHostRegister; with UVA the host pointer itself).  All tensor pointers must be
 *    16-byte aligned (ids: 4-byte).
 *  - bf16 = raw upper 16 bits of an IEEE fp32, row-major, innermost dimension contiguous.
 *  - Shapes use B batch, Hq query heads, Hkv KV heads (= GQA groups), G = Hq/Hkv, R = B*Hkv rows,
 *    D head dim (= Forecast width), S block size (64), Nb blocks per row, k = topk.
 *    KV cache / host_kv : [R][Nb][2][S][D] bf16, plane 0 = K, plane 1 = V: one block's K+V is one
 *                         contiguous 2*S*D*2-byte run (32 KiB at D=128).
 *    dev_pool           : [R][k][2][S][D] bf16, slot i of row r holds block ids[r][i].
 *    Kpool              : [R][Nb][D] bf16, one mean-pooled key per block (Eq.2, kernel=stride=S).
 *    F                  : [R][D] bf16, one Forecast head per GQA group.
 *    Q, O               : [B][Hq][D] bf16; head h belongs to group h / G.
 *    ids                : [R][k] int32, ascending block ids, -1 padded.
 *  - Ownership: the caller owns every tensor and every stream; the library owns only the workspace
 *    allocated by sparda_create (split-K partials, tickets, events).  No call
 *    allocates after sparda_create, synchronises the host, or copies results to the host.
 *  - `stream` arguments are cudaStream_t values passed as void* (torch: stream.cuda_stream).  Calls on
 *    one context must be issued from one host thread at a time.  Work is enqueued asynchronously; a
 *    return of SPARDA_OK means "enqueued", errors of the kernels themselves surface at the next CUDA
 *    synchronisation.
 *  - Errors: negative return codes below; sparda_strerror() names them, sparda_last_cuda_error() returns
 *    the CUDA error text of the last SPARDA_ECUDA on the calling context.  There is no CPU fallback
 *    and no other backend: on a device that is not sm_100 sparda_create returns SPARDA_EUNSUPPORTED.
 */
#ifndef SPARDA_H_
#define SPARDA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPARDA_OK 0
#define SPARDA_EINVAL (-1)       /* null / misaligned pointer, shape outside the supported set */
#define SPARDA_EUNSUPPORTED (-2) /* device is not sm_100 (B200) */
#define SPARDA_ECUDA (-3)        /* a CUDA runtime / driver call failed; see sparda_last_cuda_error */
#define SPARDA_ENOMEM (-4)       /* workspace allocation failed in sparda_create */
#define SPARDA_ELIMIT (-5)       /* shape beyond the fixed capacity of sparda_sparse_decode_noalloc's built-in scratch array */

#define SPARDA_GATHER_TMA 0 /* persistent single-thread-per-CTA bulk-copy (TMA) ring: host -> smem -> HBM */
#define SPARDA_GATHER_LDG 1 /* persistent warps issuing 16-byte vector loads from mapped host memory */

typedef struct sparda_ctx sparda_ctx; /* opaque */

typedef struct {
    int batch;       /* B  >= 1 */
    int n_q_heads;   /* Hq, multiple of n_kv_heads; G = Hq/Hkv in {1,2,4,8,16} */
    int n_kv_heads;  /* Hkv */
    int head_dim;    /* D in {64, 128} */
    int block_size;  /* S, must be 64 */
    int max_blocks;  /* largest Nb any call will pass (<= 8192) */
    int topk;        /* largest k any call will pass (<= 256) */
    int gather_ctas; /* persistent gather grid size; 0 = default (8 for TMA, 16 for LDG: alone on the link 2 TMA CTAs reach the
                        plateau, but beside a kernel that saturates HBM the read latency triples and 4 CTAs deliver 34 GB/s
                        where 8 deliver 49; bench.py gather_sweep has the B200 trade-off between link rate, rate under
                        load and what the CTAs cost the compute stream; Table 7)                            */
    int gather_mode; /* SPARDA_GATHER_TMA or SPARDA_GATHER_LDG */
    int attn_splits; /* split-K CTAs per row for sparse_decode; 0 = auto from B, Hkv, k and the SM count */
    int max_layers;  /* largest n_layers sparda_decode_step will see (events are pre-created); 0 = 64 */
    int select_cluster; /* CTAs per row (thread-block cluster size) of forecast_select: 0 = auto from B, Hkv, n_cand and the
                           SM count; 1, 2, 4, 8 or 16 forces it (sweeps and tests)                                       */
    int hidden;      /* model width of the optional in-step Forecast projection (sparda_layer.X / .WF); 0 = not used;
                        else a multiple of 64 in [64, 8192]                                                              */
    int attn_impl;   /* 0 = sparse_decode on mma.sync (default); 1 = the tcgen05 "swap-AB" experiment (tokens on the M side,
                        accumulators in TMEM) for D = 128 and row-aligned splits, anything else falls back to 0          */
    int no_pdl;      /* 0 = the stand-alone calls and the serial step launch their kernels with programmatic dependent
                        launch: a kernel's launch and prologue overlap the tail of the previous kernel of the stream, and
                        forecast_select also streams pooled keys into its ring before that kernel has completed.  This
                        is transparent behind any kernel that does not signal launch completion early (pool_keys,
                        append_kv, anything of the caller's that does not execute griddepcontrol.launch_dependents): the
                        dependent then starts after it has completed.  libsparda's kernels that do signal early never
                        write pooled keys.  A caller whose own kernel signals early AND writes Kpool right before a
                        select must set 1.  1 = plain launches (also: what the launch gap costs).                       */
} sparda_config;

/* One decoder layer's tensors for sparda_decode_step (Algorithm 2). */
typedef struct {
    const void* F;     /* [R][D] device.  Forecast produced in this layer; selects B_{l+1}.  Unused for
                          the last layer.                                                            */
    const void* Q;     /* [B][Hq][D] device.                                                                   */
    const void* Kpool; /* [R][Nb][D] device: this layer's pooled keys (kept on GPU).            */
    const void* kv;    /* this layer's KV cache [R][Nb][2][S][D]: layer 0 = device pointer (layer-0 cache stays
                          on GPU); layers >= 1 = host-mapped pointer (pinned CPU memory) */
    void* O;           /* [B][Hq][D] device, written.                                                          */
    int32_t* ids;      /* [R][k] device, written: B_l.                                                         */
    /* Optional: Alg.2 l.1's share of the path, the Forecast projection (Eq.3).  When X and WF are non-NULL the step
     * computes F = bf16(X . WF) into the buffer F points to (which is then written, not read) with
     * sparda_forecast_project's kernel, on the stream and just before the selection that reads it; cfg.hidden must be set.
     * WFcur: layer 0 only, the extra same-layer projection F_0^cur, written to the step's F0cur buffer.     */
    const void* X;     /* [B][hidden] device, this layer's input hidden states; NULL = F is an input                  */
    const void* WF;    /* [hidden][Hkv*D] device                                                                       */
    const void* WFcur; /* [hidden][Hkv*D] device, layer 0 only                                                         */
} sparda_layer;

#define SPARDA_STEP_OVERLAP 0    /* gather on prefetch_stream, overlapped with the compute stream (the method) */
#define SPARDA_STEP_SERIAL 1     /* same kernels, everything on compute_stream in Algorithm-2 order (no overlap) */

/* Create a context for one shape family on the current device.  Allocates the workspace (split-K partials
 * R*max_splits*16*(D+2) floats, R tickets, 3*max_layers events, an internal select stream, host-step staging, a 256
 * KiB-per-SM score tile for the comparison selector).  Launcher state (shared-memory opt-ins, cluster occupancy answers,
 * the TMA descriptor cache) lives in the context: contexts of different shapes and devices coexist in one process.
 * Returns SPARDA_OK, SPARDA_EINVAL, SPARDA_EUNSUPPORTED, SPARDA_ENOMEM or SPARDA_ECUDA; *out is set only on
 * success.  Destroy with sparda_destroy (synchronises the device first).                                     */
int sparda_create(const sparda_config* cfg, sparda_ctx** out);
int sparda_destroy(sparda_ctx* ctx);

/* (a0) Key compression, Eq.2 with kernel = stride = S: Kpool[r,j,:] = bf16(mean_t K[r,j,t,:]),
 * fp32 sum in ascending t, one rounding.  kv: device pointer to [R][n_blocks][2][S][D] (a staged chunk of the
 * cache); kpool: device [R][n_blocks][D].  n_rows may be any positive count (not tied to the context's R).
 * Pre-condition of the path ("kept on GPU and updated incrementally"), not on the timed path.  */
int sparda_pool_keys(sparda_ctx* ctx, const void* kv, int64_t n_rows, int n_blocks, void* kpool, void* stream);

/* (A4 / f4) Forecast projection, Eq.3: F[b, g, :] = bf16(X[b, :] . W_F[:, g*D:(g+1)*D]), one Forecast head of
 * width D per GQA group; fp32 accumulation in a fixed order (deterministic), one rounding.  X [B][hidden] device bf16 (the
 * layer's input hidden states), W_F [hidden][Hkv*D] device bf16 row-major, F_out [R][D] device (R = B*Hkv, the layout
 * sparda_forecast_select reads).  64 <= hidden <= 8192, a multiple of 64.  One kernel on `stream` (cluster split-K on
 * mma.sync, partials reduced in a fixed order through distributed shared memory; no workspace); bound by streaming W_F
 * once.  The path's calls take F as an input, so a caller that computes F inside its fused QKV+F GEMM does not need this;
 * sparda_layer.X / .WF run it inside sparda_decode_step.                                                                */
int sparda_forecast_project(sparda_ctx* ctx, const void* X, const void* WF, int hidden, void* F_out, void* stream);

/* (f2) Decode-time cache maintenance, Alg.2 lines 2-3: append the new token's key and value at position t
 * (0-based; block t / S, offset t % S) of every row's cache and "update K~ incrementally".  k_new, v_new
 * [R][D] device; kv_cache [R][n_blocks][2][S][D]: a device pointer (layer 0) or a host-mapped pointer (the offloaded
 * layers: the 2*D*2 bytes per row are written through UVA, the asynchronous CPU write-back of P:L159); ksum [R][D] fp32
 * device, owned by the caller, zero-initialised, carried from call to call: the running fp32 sum of the open block's
 * keys in arrival order; kpool [R][n_blocks][D] device: row j is written when t % S == S - 1, bit-identical to
 * sparda_pool_keys on the finished block, and ksum is reset.  Tokens must be appended in ascending t.  The candidate
 * range of the next selection is the complete blocks, n_cand = (t + 1) / S.  One small kernel on `stream`.          */
int sparda_append_kv(sparda_ctx* ctx, const void* k_new, const void* v_new, int64_t t, void* kv_cache, int n_blocks,
                     float* ksum, void* kpool, void* stream);

/* (a1+a2) Forecast indexer, Eq.4: s[r,j] = sum_d F[r,d]*Kpool[r,j,d] (raw logits, fp32
 * accumulate, no softmax, no scale) for candidate blocks j in [0, n_cand); ids_out[r] = the min(topk, n_cand)
 * best blocks, ties to the lowest block id, emitted in ascending block id and padded with -1.
 * F [R][D], Kpool [R][n_blocks][D], ids_out [R][topk]: device.  0 <= n_cand <= n_blocks <= max_blocks,
 * 1 <= topk <= cfg.topk.  One kernel launch on `stream` (one thread-block cluster per row; the scores stay in
 * shared memory).                                                                                              */
int sparda_forecast_select(sparda_ctx* ctx, const void* F, const void* Kpool, int n_blocks, int n_cand, int topk,
                           int32_t* ids_out, void* stream);

/* (a3) Prefetch launch, Alg.2 l.5, Sec.4.3: one persistent kernel on `stream` (the prefetch
 * stream) copies, for every (r, i) with ids[r][i] >= 0, the 2*S*D*2 bytes of block ids[r][i] of host_kv
 * [R][n_blocks][2][S][D] (host-mapped; a device pointer also works) to slot i of dev_pool [R][topk][2][S][D].
 * ids is a DEVICE pointer read when the kernel runs, so the launch can be enqueued before the selection has
 * executed; the caller orders it after the select and before the attention with events.  Slots whose id is -1
 * are left untouched.  Exact byte copy.                                                                       */
int sparda_prefetch_launch(sparda_ctx* ctx, const void* host_kv, int n_blocks, const int32_t* ids, int topk,
                           void* dev_pool, void* stream);

/* (f4, outside the paper) Peer-HBM offload tier: the KV cache of the offloaded layers may live in another GPU's HBM instead
 * of pinned host memory -- same block layout, same persistent gather, the loads travel over NVLink / NVSwitch instead of
 * PCIe.  sparda_prefetch_launch takes any pointer the current device can dereference; this call makes
 * `peer_device`'s memory such a pointer (cudaDeviceEnablePeerAccess from the context's device; calling it again is not an
 * error).  The link's bandwidth-delay product is ~30 times PCIe's, so give the gather more CTAs on this tier
 * (cfg.gather_ctas; bench.py roofline.gather_sweep.hbm_tier has the engine's rate by CTA count with the link out of the way).
 * Returns SPARDA_EUNSUPPORTED when the two devices have no peer path, SPARDA_EINVAL for peer_device == the context's device
 * or out of range.  Host-synchronous (driver call); not for the decode loop.                                            */
int sparda_enable_peer_tier(sparda_ctx* ctx, int peer_device);

/* (a5/a6) Block-sparse GQA attention with the real query, Eq.5, Alg.2 l.7:
 * O[b,h,:] = bf16( softmax_t( q_h . k_t / sqrt(D) ) V ) over every token t of every selected block of row
 * r = b*Hkv + h/G; bf16 tensor-core products, fp32 softmax and accumulation, one rounding; no causal mask
 * inside a block (the query sits after the context).  Slots with id -1 are skipped; a row with no valid slot
 * gives O = 0.
 *   pool_is_indexed = 0: dev_pool is [R][topk][2][S][D] and slot i holds block ids[r][i] (n_slots = topk);
 *   pool_is_indexed = 1: dev_pool is a device-resident cache [R][n_slots][2][S][D] addressed through ids
 *                        (layer 0).
 * Split-K flash-decode over a flat list of the R*topk slots.  Row-aligned splits with 2, 4, 8 or 16 CTAs per row run as
 * one thread-block cluster per row and reduce their partials through distributed shared memory; any other split
 * reduces through the context's L2-resident workspace, merged by the last CTA of each row (ticket).
 * The workspace is shared by every launch on the context: at most ONE sparse_decode may be in flight per context at a
 * time -- order concurrent launches with events or use one context per stream.  (The other kernels keep their
 * intermediate state in shared memory and may overlap freely.)                                                  */
int sparda_sparse_decode(sparda_ctx* ctx, const void* Q, const void* dev_pool, const int32_t* ids, int topk,
                         int pool_is_indexed, int n_slots, void* O, void* stream);

/* (a5/a6 + f2) The same attention over caches whose newest block is partly filled (reading q7).  Alg.2 l.2 appends the
 * new token's K / V before the attention and Eq.1 always attends the local window that holds it, so a row's cache
 * holds seq_len[r] tokens and its last block min(S, seq_len[r] - S*j) of them.  seq_len: device [R] int32.  For every listed
 * block id j >= 0 of row r only its first min(S, seq_len[r] - S*j) tokens are attended; a block with none (S*j >= seq_len[r])
 * counts like id -1.  Whatever bytes lie behind the last token of the open block are ignored (NaN included: their scores are
 * replaced, their V rows zeroed in shared memory), so the cache need not be cleared.  ids holds BLOCK ids in both pool forms
 * (with pool_is_indexed = 0, slot i of dev_pool holds block ids[r][i] as for sparda_sparse_decode).  The caller lists the open
 * block itself: the selectors rank complete blocks only (sparda_set_step_candidates), so append its id (the highest: the
 * list stays ascending) to the selection, gather it like any other block (sparda_append_kv has written it to the host cache), or
 * attend a device-resident cache by id.  Every other rule, and the one-launch-per-context limit, as for sparda_sparse_decode.
 * The decode steps do not pass seq_len yet: they attend complete blocks only.                                                */
int sparda_sparse_decode_varlen(sparda_ctx* ctx, const void* Q, const void* dev_pool, const int32_t* ids, const int32_t* seq_len,
                                int topk, int pool_is_indexed, int n_slots, void* O, void* stream);

/* (a5/a6) The same attention for callers that must not allocate device memory, and so cannot use sparda_create at all
 * (it calls cudaMalloc for the split-K workspace, creates a stream and events).  Who that is:
 *   - a serving engine that hands the whole of HBM to its own pool at start-up: a later cudaMalloc from a library fails,
 *     or takes memory the engine's accounting believes it owns;
 *   - a latency-critical decode loop that cannot afford the device-wide synchronisation cudaMalloc / cudaFree imply;
 *   - a plug-in or custom op that is handed pointers and a stream and has no start-up or shut-down hook in which a
 *     context could be created and destroyed.
 * This call takes no context.  Same kernel as sparda_sparse_decode (the flat split-K form, CTA partials merged by the
 * last CTA of each row), same arguments and layouts; the shape that a context would carry is passed as plain integers.
 * The split-K partials and the per-row tickets live in ONE fixed array compiled into the library
 * (SPARDA_NOALLOC_SCRATCH_BYTES = 4 260 864 bytes, about 4.1 MiB): every GPU on which the process loads libsparda holds
 * that much from module load until the process exits, whether or not this call is ever made.
 *   Limits: R = batch * n_kv_heads <= SPARDA_NOALLOC_MAX_ROWS (256); the CTAs-per-row split is chosen so that R * (partials
 *   per row) <= SPARDA_NOALLOC_MAX_PARTIALS (512), which every R within the limit allows.  A larger R returns SPARDA_ELIMIT
 *   and sparda_noalloc_last_error() names the limit.  Other shape rules are sparda_create's (G in {1,2,4,8,16},
 *   head_dim in {64,128}, topk <= 256, n_slots <= 8192; pool_is_indexed = 0 requires n_slots == topk): SPARDA_EINVAL.
 *   Set-up: the FIRST call on each device (with that device current, as for every call) resolves the device address of the
 *   array, the TMA descriptor encoder and the kernel's shared-memory opt-in; make that first call during start-up, before
 *   any stream capture begins.  Neither the first nor any later call calls cudaMalloc, cudaFree or any routine that
 *   allocates device memory; the only extra work enqueued on `stream` is a cudaMemsetAsync of the R tickets in front of the
 *   kernel (the array keeps whatever the previous call left, the tickets must start at zero).
 *   Sharing: every call on a device uses the same array.  Two calls that can run on the GPU at the same time (different
 *   streams without an event between them) race on it and give wrong output; calls on one stream are safe.  Host side, the
 *   call is serialised by a lock and may be made from any thread.
 * Returns SPARDA_OK (enqueued), SPARDA_EINVAL, SPARDA_ELIMIT, SPARDA_EUNSUPPORTED (not an sm_100 device) or SPARDA_ECUDA;
 * sparda_noalloc_last_error() returns the calling thread's last failure of this entry point as text ("" if none).  */
#define SPARDA_NOALLOC_MAX_ROWS 256
#define SPARDA_NOALLOC_MAX_PARTIALS 512
#define SPARDA_NOALLOC_SCRATCH_BYTES (SPARDA_NOALLOC_MAX_PARTIALS * (16 * 128 * 4 + 2 * 16 * 4) + SPARDA_NOALLOC_MAX_ROWS * 4)
int sparda_sparse_decode_noalloc(int batch, int n_q_heads, int n_kv_heads, int head_dim, const void* Q, const void* dev_pool,
                                 const int32_t* ids, int topk, int pool_is_indexed, int n_slots, void* O, void* stream);
const char* sparda_noalloc_last_error(void);

/* (a4 + a6) One decode step over n_layers layers in Algorithm-2 order with the one-layer-ahead
 * pipeline: layer 0 selects with F0cur against its own Kpool and attends straight from its device-resident
 * cache; for l >= 1, ids_l = f_top(F_{l-1} Kpool_l^T) is selected during layer l-1, gathered
 * into dev_pool[l & 1] on prefetch_stream and attended in layer l after an event wait.  The pool is
 * double-buffered: gather l+1 may start only after attention l-1 released its buffer.
 * mode = SPARDA_STEP_OVERLAP or SPARDA_STEP_SERIAL (same kernels on one stream; results are bit-identical).
 * In overlap mode a layer's gather is launched together with its select and waits on the device for the select's
 * doorbell (one counter per layer in the context's workspace, zeroed at the top of the step), so no kernel boundary
 * sits between "block list out" and "first byte on the link"; a gather whose select never runs traps after ~15 s
 * instead of hanging the device.  The doorbell is used only while the gather grid cannot fill the device (cfg.gather_ctas <=
 * SM count / 2 = 74 on B200: the select can then always become resident beside the waiting CTAs, also in a graph replay where
 * nothing orders the two launches); a larger gather grid is launched behind the select's event instead (same results, one kernel
 * boundary more on the chain).  One step per context at a time.  The select runs on a highest-priority stream of the
 * context; create prefetch_stream with the highest priority too (cudaStreamCreateWithPriority): beside a many-CTA kernel on
 * the compute stream the block scheduler serves the older kernel's pending CTAs first, and at equal priority a side-stream
 * kernel launched after it waits for most of it (measured: select 42 us instead of 20 beside a 4736-CTA HBM stream).
 * Capturable into a CUDA graph (no host synchronisation, events are pre-created).                             */
int sparda_decode_step(sparda_ctx* ctx, const sparda_layer* layers, int n_layers, const void* F0cur, int n_blocks,
                       int topk, void* dev_pool0, void* dev_pool1, void* compute_stream, void* prefetch_stream,
                       int mode);

/* Growing caches (Alg.2 l.2-3): a cache allocated for n_blocks blocks holds t + 1 tokens, of which
 * n_cand = (t + 1) / S blocks are complete and have a pooled key (sparda_append_kv).  After this call the selections of
 * sparda_decode_step / _host / _cached rank blocks [0, n_cand) only (n_blocks stays the layout stride); 0 restores
 * n_cand = n_blocks.  With n_cand <= topk every complete block is selected and the rest of the ids is -1 (reading q5).
 * Host-side state of the context: set it before the step is enqueued (or captured).                              */
int sparda_set_step_candidates(sparda_ctx* ctx, int n_cand);

/* (f3 inside a4) The paper's selector geometry in the decode steps: after sparda_set_step_selector(ctx, 1, n_init, n_local)
 * every selection of sparda_decode_step / _host / _cached is sparda_forecast_select_grid -- layers[l].Kpool then points to the
 * (32,16) compressed-key grid [R][4 n_blocks][D] of sparda_pool_keys_grid, and ids are init + local + top-k (Eq.1, P:L53;
 * reading q19: parity unpinned by the paper).  n_init + n_local <= topk.  grid = 0 restores the one-key-per-block form.
 * The cached step then runs the reuse plan as its own launch behind the select (no doorbell for that layer's gather).
 * With a growing cache (sparda_set_step_candidates): sparda_append_kv maintains only the one-key-per-block Kpool, NOT the grid.
 * The four grid keys of a block exist only after sparda_pool_keys_grid has run over it, so a caller that combines grid = 1 with a
 * growing n_cand must re-run sparda_pool_keys_grid over every newly completed block (and, because the (32,16) windows straddle
 * block boundaries, over the block before it) before the step that first ranks it; otherwise that block is ranked on stale or
 * zero keys.  Nothing in the library detects this.                                                                          */
int sparda_set_step_selector(sparda_ctx* ctx, int grid, int n_init, int n_local);

/* The same step for a caller whose per-step tensors live in HOST memory (the end-to-end form bench.py times):
 * layers[l].F, .Q and .O and F0cur are HOST pointers (pinned for the copies to be asynchronous); the call runs
 * sparda_decode_step on staging owned by the context and enqueues the copies on compute_stream just in time: F0cur first,
 * F_l and Q_l before layer l begins, O_l right after attention l -- so they run while that stream waits for a gather.
 * layers[l].Kpool, .kv and .ids keep their sparda_decode_step meaning.  No host synchronisation: O is valid once
 * compute_stream has drained.  Needs n_layers <= max_layers.                                                   */
int sparda_decode_step_host(sparda_ctx* ctx, const sparda_layer* layers, int n_layers, const void* F0cur, int n_blocks,
                            int topk, void* dev_pool0, void* dev_pool1, void* compute_stream, void* prefetch_stream,
                            int mode);

/* (f1) Step-to-step block reuse.  The paper's engine keeps, per layer, the blocks selected at the previous decode
 * step and fetches "only newly selected blocks" (App. C); it states no slot policy, so this library fixes one
 * (reading q18): a pool slot whose block is selected again keeps it; the j-th smallest newly selected block
 * that is not resident goes to the j-th lowest-numbered slot whose block was not selected again; slots left over
 * become empty (-1).
 *   ids_new  [R][topk] device, this step's selection as written by sparda_forecast_select (ascending, -1 padded);
 *   slot_ids [R][topk] device, in/out: the block each slot of the layer's persistent pool holds (-1 = empty; the
 *            caller initialises it to -1 once);
 *   fetch    [R][topk] device, out: fetch[r][s] = block to copy into slot s, or -1 -- pass it as `ids` to
 *            sparda_prefetch_launch; pass slot_ids as `ids` to sparda_sparse_decode (pool_is_indexed = 0);
 *   n_fetch  [R] device, out (may be NULL): blocks to fetch per row.
 * One small kernel on `stream`; topk <= 256.                                                                  */
int sparda_reuse_plan(sparda_ctx* ctx, const int32_t* ids_new, int topk, int32_t* slot_ids, int32_t* fetch,
                      int32_t* n_fetch, void* stream);

/* (f3) The paper's selector geometry.  PARITY UNPINNED BY THE PAPER: Eq.2 with (l_C, s) = (32, 16) fixes
 * the compressed keys, but the max-pool that turns compressed-grid scores into block scores has no stated
 * kernel, stride or padding; this library takes reading q19.
 * sparda_pool_keys_grid: Kgrid[r, j, :] = bf16(mean of keys 16 j .. 16 j + 31), fp32 sum in ascending token order,
 *   j < 4 * n_blocks - 1; kv [R][n_blocks][2][S][D] device, kgrid [R][4 * n_blocks][D] device (last row zero).
 * sparda_forecast_select_grid: s_j = F[r] . Kgrid[r, j] (raw logits, Eq.4); block b's score = max of s_j over the
 *   compressed keys whose window starts inside the block, j = 4b .. 4b+3 with j < 4 * n_cand - 1 (f_top); blocks
 *   [0, n_init) (initial) and [n_cand - n_local, n_cand) (local window) are always selected and do not compete (Eq.1,
 *   P:L53); the remaining topk - n_init - n_local places go to the best other candidates, ties to the lowest id;
 *   ids_out [R][topk] ascending, -1 padded.  The paper's budget is topk = 96 = 1 + 32 + 63.              */
int sparda_pool_keys_grid(sparda_ctx* ctx, const void* kv, int64_t n_rows, int n_blocks, void* kgrid, void* stream);
int sparda_forecast_select_grid(sparda_ctx* ctx, const void* F, const void* Kgrid, int n_blocks, int n_cand, int n_init,
                                int n_local, int topk, int32_t* ids_out, void* stream);

/* sparda_forecast_select followed by sparda_reuse_plan on its result, in ONE launch: the CTA that selects a row also
 * updates the row's slot table and fetch list (same results as the two calls; saves a launch per layer of the cached
 * decode step).  Arguments as in the two calls.                                                                   */
int sparda_forecast_select_plan(sparda_ctx* ctx, const void* F, const void* Kpool, int n_blocks, int n_cand, int topk,
                                int32_t* ids_out, int32_t* slot_ids, int32_t* fetch, int32_t* n_fetch, void* stream);

/* One decoder layer of sparda_decode_step_cached: sparda_layer plus the layer's persistent pool and slot table.   */
typedef struct {
    sparda_layer base;   /* as in sparda_decode_step                                                             */
    void* pool;          /* [R][topk][2][S][D] device, owned by the caller, persistent across steps (layer 0: unused) */
    int32_t* slot_ids;   /* [R][topk] device, in/out (see sparda_reuse_plan); initialise to -1                   */
    int32_t* fetch;      /* [R][topk] device, written                                                            */
    int32_t* n_fetch;    /* [R] device, written; may be NULL                                                     */
} sparda_cached_layer;

/* sparda_decode_step with the previous step's blocks kept per layer: per layer l >= 1 the compute stream
 * runs select B_{l+1} + reuse plan (one launch) -> [prefetch stream: gather only the missing blocks into layer l+1's own pool] ->
 * wait for layer l's gather -> attention over pool_l in slot order.  Layer 0 attends from its resident cache as
 * before.  Same modes, same capture rules; with every slot_ids at -1 the step moves exactly the bytes of
 * sparda_decode_step.                                                                                           */
int sparda_decode_step_cached(sparda_ctx* ctx, const sparda_cached_layer* layers, int n_layers, const void* F0cur,
                              int n_blocks, int topk, void* compute_stream, void* prefetch_stream, int mode);

/* Per-kernel device timing of sparda_decode_step (measurement aid).  While enabled, every kernel
 * launched by sparda_decode_step is bracketed by timing events on the stream it is launched on (after any
 * stream wait, so a wait is not counted).  sparda_profile_read synchronises on those events and returns, for
 * kind 0 = select, 1 = gather, 2 = attention, the summed milliseconds and launch counts of the LAST
 * sparda_decode_step call.  Not capturable into a CUDA graph while enabled.                                   */
int sparda_profile_enable(sparda_ctx* ctx, int on);
int sparda_profile_read(sparda_ctx* ctx, double ms_out[3], int64_t count_out[3]);

/* (a7) Chunked-prefill selection with the Forecast indexer, Alg.1 l.2: for query positions
 * i = row0 .. row0+n_rows-1 of every group g, scores = F[g,i,:] . Kpool[g,j,:] for the causal candidates
 * j < (i+1)/S (a block is visible once its last token <= i), top-k as in forecast_select.
 * F [Hkv][T][D], Kpool [Hkv][n_blocks][D], ids_out [Hkv][n_rows][topk]: device.  Dense bf16 contraction on
 * tcgen05 tensor cores (fp32 accumulators in TMEM) with a fused per-row top-k epilogue; scores never leave the
 * SM.  Supported: n_blocks <= 512 (one 128 x 512 fp32 accumulator fills TMEM), topk <= 64, else SPARDA_EINVAL.
 * Chunking: any [row0, row0 + n_rows) inside [0, T); one launch per call.                                     */
int sparda_prefill_select(sparda_ctx* ctx, const void* F, const void* Kpool, int T, int n_blocks, int row0,
                          int n_rows, int topk, int32_t* ids_out, void* stream);

/* (a7') The comparison selector (Eq.6 left term): per query head h of group g,
 * softmax_j(Q[h,i,:] . Kpool[g,j,:] / sqrt(D)) over the same causal candidates, summed over the G heads,
 * then the same top-k.  Q [Hq][T][D] device.                                                                  */
int sparda_prefill_select_baseline(sparda_ctx* ctx, const void* Q, const void* Kpool, int T, int n_blocks, int row0,
                                   int n_rows, int topk, int32_t* ids_out, void* stream);

/* Measurement aids, NOT part of the method (csrc/bench_probes.cu).
 * sparda_probe_launch enqueues one probe kernel on `stream`: kind 0 = empty kernel (launch floor); 1 = empty kernel with
 * the forecast_select launch shape (128 CTAs x 288 threads, clusters of 2, 107 KB of shared memory); 2 = 148 CTAs, one
 * dependent DRAM load each (buf: device, bytes >= 148 MiB, untouched locations 1 MiB apart); 3 = the layer stand-in:
 * streams `bytes` of buf (device, 16-byte aligned) from HBM once.
 * sparda_set_layer_standin(ctx, weights, bytes): while bytes > 0, sparda_decode_step[_cached|_host] launches the stand-in
 * on the compute stream after every attention -- the cost of the rest of a decoder layer (an 8B layer reads ~474 MB of
 * bf16 weights per token step: o-proj, FFN, the next QKV+F projections), so that "gather hidden behind
 * the next layer's compute" can be measured.  bytes = 0 switches it off (the default).                       */
int sparda_probe_launch(sparda_ctx* ctx, int kind, const void* buf, int64_t bytes, void* stream);
int sparda_set_layer_standin(sparda_ctx* ctx, const void* weights, int64_t bytes);

/* Introspection used by bench.py / tests: number of kernels this context has launched since creation, the
 * resolved tunables, and error text.                                                                          */
int64_t sparda_launch_count(const sparda_ctx* ctx);
int64_t sparda_tmap_encodes(const sparda_ctx* ctx);      /* TMA descriptors encoded so far (a warm step encodes none) */
int sparda_get_select_cluster(const sparda_ctx* ctx);    /* cluster size of the LAST forecast_select launch           */
int sparda_get_attn_cluster(const sparda_ctx* ctx);      /* CTAs per row reduced through DSMEM by the LAST sparse_decode
                                                            launch (2, 4, 8, 16), 0 = workspace + ticket reduction      */
int sparda_get_attn_splits(const sparda_ctx* ctx, int topk);
int sparda_get_gather_ctas(const sparda_ctx* ctx);
const char* sparda_strerror(int code);
const char* sparda_last_cuda_error(const sparda_ctx* ctx);
const char* sparda_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPARDA_H_ */
