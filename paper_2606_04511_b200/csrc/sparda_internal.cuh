// Internal declarations shared by the libsparda translation units (sm_100a only).
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/sparda.h"

#define SPARDA_TMAP_SLOTS 256   // hashed tensor-map cache (power of two): a 32-layer step presents ~64 distinct bases
#define SPARDA_MAX_G 16        // query heads per group, padded to the M=16 of mma.m16n8k16
#define SPARDA_MAX_CLUSTER 16

// Per-context launcher state of one kernel instantiation (the context lives on one device, so "per context" is also
// "per device"): whether the dynamic-shared-memory / cluster opt-in attributes have been set, and how many clusters of
// each size the device can keep resident at the shared-memory size the context uses (0 = not asked, -1 = none).
struct sparda_kernel_state {
    bool attr_set;
    int max_clusters[SPARDA_MAX_CLUSTER + 1];
    int asked_smem[SPARDA_MAX_CLUSTER + 1];   // dynamic shared memory the answer in max_clusters[] was asked for
};
enum {
    SPARDA_K_SELECT_128, SPARDA_K_SELECT_64, SPARDA_K_SELECT_GRID_128, SPARDA_K_SELECT_GRID_64,
    SPARDA_K_ATTN_128, SPARDA_K_ATTN_64, SPARDA_K_ATTN_CL_128, SPARDA_K_ATTN_CL_64,
    SPARDA_K_ATTN_VL_128, SPARDA_K_ATTN_VL_64, SPARDA_K_ATTN_VL_CL_128, SPARDA_K_ATTN_VL_CL_64,   /* sparda_sparse_decode_varlen */
    SPARDA_K_GATHER_TMA, SPARDA_K_PROBE, SPARDA_K_STANDIN, SPARDA_K_PROJECT, SPARDA_K_ATTN_T5, SPARDA_K_ATTN_T5_CL,
    SPARDA_K_PF_0, /* 8 prefill instantiations: D x BASELINE x REPL */
    SPARDA_K_COUNT = SPARDA_K_PF_0 + 8
};

struct sparda_tmap_entry {
    const void* base;
    uint64_t rows;
    int head_dim;
    int box_rows;
    CUtensorMap map;
};

struct sparda_ctx {
    sparda_config cfg;
    int sm_count;
    int R;             // B * Hkv
    int G;             // Hq / Hkv
    int max_splits;    // partial slots per row in the workspace
    // workspace (device)
    float* part_O;     // [R][max_splits][16][D]
    float* part_ml;    // [R][max_splits][2][16]  (m in log2 domain, l)
    unsigned int* tickets;  // [R]: split-K attention, one per row (the select keeps its scores on chip)
    float* pf_scratch;      // prefill comparison selector: [sm_count][512][128] fp32 group-summed scores (lazy)
    cudaEvent_t* ev_sel;    // [max_layers + 1]
    cudaEvent_t* ev_gather; // [max_layers + 1]
    cudaEvent_t* ev_top;    // [max_layers + 1]: layer l may begin (attention l-1 is enqueued before it on the compute stream)
    cudaStream_t select_stream;  // internal: select B_{l+1} runs here, concurrently with attention l (decode_step, overlap mode)
    int max_layers;
    // host-buffer step staging (device): F [(max_layers+1)][R][D] (slot max_layers = F0cur), Q and O [max_layers][B][Hq][D]
    char* stage_F;
    char* stage_Q;
    char* stage_O;
    // per-kernel timing of sparda_decode_step: events [kind 0..2][max_layers + 1][start, stop]
    int prof_on;
    cudaEvent_t* ev_prof;
    int prof_n[3];
    int64_t launches;
    int last_select_cluster, last_attn_cluster;   // introspection: the shape the last launch resolved to
    // Programmatic dependent launch for the NEXT launch (cfg.no_pdl overrides): 1 for the stand-alone calls and for the
    // serial step (one stream, kernel after kernel: 0.60 ms per cached batch-4 step against 0.68 without); 0 inside an
    // overlapped step, where every chain starts behind an event wait and early-resident dependents only take shared memory
    // from the kernels of the other streams (measured: 0.43 ms with PDL on the in-chain launches, 0.38 ms without)
    int pdl_next;
    // Doorbells between the select and the gather of a layer inside the overlapped step (sparda_api.cu): door[l] counts the rows
    // of layer l whose block list is out in this step (zeroed at the top of every step).  door_next != nullptr: the NEXT select
    // / gather launch rings / waits on it (the step sets it; stand-alone calls never do).
    unsigned int* door;       // [max_layers + 1]
    unsigned int* door_next;
    int step_grid, step_n_init, step_n_local;   // sparda_set_step_selector: the steps select with the (32,16) grid form (f3)
    int step_n_cand;          // sparda_set_step_candidates: blocks [0, step_n_cand) are ranked by the decode steps (0 = all n_blocks)
    char cuda_err[256];
    // TMA descriptor cache (host): open-addressed hash on (base, rows, head_dim, box_rows); lookups return a COPY, so an
    // eviction can never change a descriptor a launcher already holds
    sparda_tmap_entry tmaps[SPARDA_TMAP_SLOTS];
    int64_t tmap_encodes;   // descriptors encoded so far (introspection: a warm step must not encode)
    void* encode_fn;   // cuTensorMapEncodeTiled
    int device;             // the device the context was created on
    // measurement aids (bench_probes.cu): a sink the probe kernels may write, and the optional layer stand-in
    uint32_t* probe_sink;   // [256]
    const void* standin_buf;
    size_t standin_bytes;
    sparda_kernel_state kstate[SPARDA_K_COUNT];
};

int sparda_set_cuda_error(sparda_ctx* ctx, cudaError_t e, const char* where);
#define SPARDA_CUDA_TRY(ctx, call)                                             \
    do {                                                                       \
        cudaError_t e__ = (call);                                              \
        if (e__ != cudaSuccess) return sparda_set_cuda_error(ctx, e__, #call); \
    } while (0)

// launch attribute that allows this launch to overlap its prologue with the tail of the previous kernel of the stream (PDL)
static inline cudaLaunchAttribute sparda_pdl_attr() {
    cudaLaunchAttribute a;
    a.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    a.val.programmaticStreamSerializationAllowed = 1;
    return a;
}

static inline bool sparda_use_pdl(const sparda_ctx* ctx) { return !ctx->cfg.no_pdl && ctx->pdl_next; }

static inline bool sparda_aligned(const void* p, uintptr_t a) { return p != nullptr && ((uintptr_t)p & (a - 1)) == 0; }

// launchers implemented in the kernel translation units
int sparda_launch_pool_keys(sparda_ctx*, const void* kv, int64_t n_rows, int n_blocks, void* kpool, cudaStream_t);
int sparda_launch_select(sparda_ctx*, const void* F, const void* Kpool, int n_blocks, int n_cand, int topk,
                         int32_t* ids, int32_t* slot_ids /* optional fused reuse plan */, int32_t* fetch, int32_t* n_fetch,
                         cudaStream_t);
int sparda_launch_gather(sparda_ctx*, const void* host_kv, int n_blocks, const int32_t* ids, int topk, void* pool,
                         cudaStream_t);
int sparda_launch_forecast_project(sparda_ctx*, const void* X, const void* WF, int hidden, void* F, cudaStream_t);
int sparda_launch_pool_keys_grid(sparda_ctx*, const void* kv, int64_t n_rows, int n_blocks, void* kgrid, cudaStream_t);
int sparda_launch_select_grid(sparda_ctx*, const void* F, const void* Kgrid, int n_blocks, int n_cand, int n_init, int n_local, int topk,
                              int32_t* ids, cudaStream_t);
int sparda_launch_append_kv(sparda_ctx*, const void* k_new, const void* v_new, int64_t t, void* kv, int n_blocks, float* ksum,
                            void* kpool, cudaStream_t);
int sparda_launch_reuse_plan(sparda_ctx*, const int32_t* ids_new, int topk, int32_t* slot_ids, int32_t* fetch, int32_t* n_fetch,
                             cudaStream_t);
int sparda_launch_attn(sparda_ctx*, const void* Q, const void* pool, const int32_t* ids, const int32_t* seq_len /* or nullptr */, int topk,
                       int indexed, int n_slots, void* O, cudaStream_t);
// the tcgen05 experiment (cfg.attn_impl = 1): SPARDA_OK, 1 = shape outside its range (fall back to the mma.sync kernel), or an error
int sparda_launch_attn_tc5(sparda_ctx*, const void* Q, const void* pool, const int32_t* ids, int topk, int indexed,
                           int n_slots, void* O, cudaStream_t);
int sparda_launch_prefill_select(sparda_ctx*, const void* F, const void* Kpool, int T, int n_blocks, int row0,
                                 int n_rows, int topk, int32_t* ids, cudaStream_t);
int sparda_launch_prefill_baseline(sparda_ctx*, const void* Q, const void* Kpool, int T, int n_blocks, int row0,
                                   int n_rows, int topk, int32_t* ids, cudaStream_t);
// [rows][head_dim] bf16 row-major view, box = box_rows x 64 elements (128 B), 128-byte swizzle; *out receives a copy
int sparda_get_tmap(sparda_ctx*, const void* base, uint64_t rows, int head_dim, int box_rows, CUtensorMap* out);
int sparda_launch_standin(sparda_ctx*, cudaStream_t);       // bench_probes.cu: the labelled layer stand-in (not the method)
int sparda_resolve_splits(const sparda_ctx*, int topk);     // average CTAs per row of the attention launch
int sparda_resolve_attn_ctas(const sparda_ctx*, int topk);  // its grid size

#ifdef __CUDACC__
// ------------------------------------------------------------------------------------------------
// Device helpers (inline PTX for sm_100a)
// ------------------------------------------------------------------------------------------------
namespace sparda {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

// ---- select -> gather doorbell (device side).  Producer: after a row's block list is in global memory (ordered before the
// calling thread by a CTA / warp barrier), one thread publishes it: the fence makes the list visible at gpu scope before the
// count.  Consumer: one thread per CTA waits until all R rows of its layer have been published.
__device__ __forceinline__ void door_ring(unsigned int* door) {
    __threadfence();
    atomicAdd(door, 1u);
}
__device__ __forceinline__ void door_wait(const unsigned int* door, unsigned int need) {
    unsigned int spins = 0;
    for (;;) {
        unsigned int v;
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(door) : "memory");
        if (v >= need) break;
        __nanosleep(64);
        if (++spins > (1u << 24)) __trap();   // ~15 s: the select this launch was paired with never ran: fail, do not hang the device
    }
}

// Programmatic dependent launch (PDL): a kernel launched with sparda_pdl_attr() may become resident and run its prologue
// (barrier init, tensor-map prefetch, index arithmetic) while the previous kernel of the stream is still draining;
// pdl_wait() blocks until that kernel has completed and its memory is visible -- it must precede every global-memory
// access -- and pdl_launch_dependents() lets the NEXT kernel do the same with this one.  Without the launch attribute both
// are no-ops.  Semantics are those of plain stream order; what is saved is the launch gap and the prologue (~1.3 us per
// kernel of a back-to-back chain on B200).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// 1-D bulk copies (TMA engine, no tensor map)
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* gdst, const void* smem_src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(smem_src)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
template <int N>
__device__ __forceinline__ void bulk_wait() {
    asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory");
}

// 2-D tiled TMA load through a tensor map (coordinates: x = innermost element index, y = row)
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int x, int y, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::
            "r"(smem_u32(smem_dst)),
        "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

__device__ __forceinline__ void ldmatrix_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2,
                                                  uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr));
}
// D(16x8, fp32) += A(16x16, bf16, row) * B(16x8, bf16, col)
__device__ __forceinline__ void mma_bf16_16816(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ float bf16_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t u) { return __uint_as_float(u & 0xFFFF0000u); }

__device__ __forceinline__ int4 ld_nc_v4(const void* p) {
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}
__device__ __forceinline__ void st_na_v4(void* p, const int4& v) {
    asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
                 "r"(v.w)
                 : "memory");
}

// order-preserving map fp32 -> uint32 (larger float <=> larger key)
__device__ __forceinline__ uint32_t orderable(float f) {
    uint32_t b = __float_as_uint(f);
    return b ^ ((b >> 31) ? 0xFFFFFFFFu : 0x80000000u);
}

}  // namespace sparda
#endif
