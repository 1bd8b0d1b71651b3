// Prefetch launch (a3): persistent UVA gather, pinned host memory -> HBM block pool.
//
// Alg.2 l.5, Sec.4.3: "a persistent ... kernel based on UVA ... keeps a small fixed set of
// CTAs active and lets them continuously process block-transfer tasks within a single launch".
//
// Task = one selected block (r, slot): 2*S*D*2 contiguous bytes at host_kv[(r*Nb + ids[r][slot])] ->
// dev_pool[(r*k + slot)].  ids are read from device memory when the kernel runs.
//
// Two engines, same tasks, same bytes:
//  * SPARDA_GATHER_TMA (default, B200-native): one warp per CTA compacts the task list and ONE of its threads drives a ring of 16 KiB shared-memory
//    stages with bulk-copy (TMA) instructions: cp.async.bulk global(host-mapped)->smem completing on an
//    mbarrier, then cp.async.bulk smem->global(HBM).  No registers or LSU slots are spent on payload, so a
//    handful of CTAs saturates the host link (measured on this box: alone on the GPU 2 CTAs x 1 thread reach the
//    50.5 GB/s plateau that takes 8+ CTAs x 256 threads with vector loads; beside a kernel that saturates HBM a
//    host read takes three times as long to come back and it takes 8 CTAs to keep 49 GB/s on the link: the
//    default), leaving the SMs to the compute stream (the trade-off of P:L116).
//  * SPARDA_GATHER_LDG: the paper's shape, persistent warps issuing 16-byte vector loads (8 in flight per
//    lane) from mapped host memory, 4 KiB per warp-iteration.
#include "sparda_internal.cuh"

namespace {

using namespace sparda;

#ifndef GATHER_STAGE_BYTES_V
#define GATHER_STAGE_BYTES_V 16384
#define GATHER_STAGES_V 6
#endif
constexpr int GATHER_STAGE_BYTES = GATHER_STAGE_BYTES_V;
constexpr int GATHER_STAGES = GATHER_STAGES_V;  // 96 KiB ring per CTA
#ifndef GATHER_PENDING_V
#define GATHER_PENDING_V 2
#endif
// Stores that may still be reading their stage when the next load is issued: the thread does not wait for each smem -> HBM
// store before it asks for the next block (loads in flight = STAGES - PENDING).  Nothing on the PCIe link (the same 50.4 GB/s with
// 0 .. 4), but from a fast source -- the peer-HBM tier -- a CTA moves more per round trip (gather_sweep.hbm_tier).
constexpr int GATHER_PENDING = GATHER_PENDING_V;

constexpr int GATHER_WIN = 1024;  // tasks compacted per window (32 per lane, held in registers)

// The task list ids[R*k] may be sparse (the reuse cache, f1, fetches only the blocks that are not resident): the warp
// first compacts the valid tasks of a window with ballots -- every CTA scans the whole window, CTA c takes the c-th
// equal share of the VALID tasks, so the split is balanced whatever the pattern -- then lane 0 drives the bulk-copy
// ring over its share.  An empty list costs one scan (a few microseconds), not one dependent load per slot.
// DOOR (overlapped decode step): the launch is already resident when the layer's select runs; it waits for the
// select's doorbell (n_rows rows published) instead of for a kernel boundary, and reads ids only after it.
//
// How ids is read depends on who wrote it.  Stream-ordered launches (DOOR = false): the list was complete before this kernel
// began and stays read-only for its lifetime, which is what the non-coherent path (ld.global.nc, __ldg) is defined for.
// DOOR = true: the select that WRITES ids runs concurrently with this kernel, so ids is not read-only over the kernel's
// lifetime; ld.global.nc would be undefined there (the compiler may treat such a load as invariant and move it above the
// door's acquire, and the acquire does not make non-coherent lines coherent).  That instantiation reads ids with ld.global.cg
// (__ldcg: coherent at L2, where the select's st + fence + atomic published it), ordered after door_wait by its "memory" clobber
// and the warp / CTA barrier.  ids carries no __restrict__ for the same reason.
template <bool DOOR>
__device__ __forceinline__ int32_t load_id(const int32_t* p) {
    if (DOOR) return __ldcg(p);
    return __ldg(p);
}

template <bool DOOR>
__global__ void __launch_bounds__(32) gather_tma_kernel(const char* __restrict__ host_kv, const int32_t* ids,
                                                        char* __restrict__ pool, int n_rows, int n_blocks, int topk,
                                                        uint32_t block_bytes, unsigned int* door) {
    extern __shared__ __align__(128) char ring[];
    __shared__ uint64_t full[GATHER_STAGES];
    __shared__ int32_t q_task[GATHER_WIN], q_id[GATHER_WIN];
    __shared__ char* dst_of[GATHER_STAGES];
    const int lane = threadIdx.x;
    if (lane == 0) {
        for (int s = 0; s < GATHER_STAGES; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
        fence_proxy_async_smem();
    }
    __syncwarp();
    pdl_wait();                  // ids (and the pool's previous reader) belong to earlier kernels
    pdl_launch_dependents();
    if (DOOR) {
        if (lane == 0) door_wait(door, (unsigned)n_rows);
        __syncwarp();
    }
    const uint32_t cpb = block_bytes / GATHER_STAGE_BYTES;  // 16 KiB chunks per block: 2 at D=128, 1 at D=64
    const int64_t n_tasks = (int64_t)n_rows * topk;
    const unsigned lt = (1u << lane) - 1u;
    int load_s = 0, store_s = 0, in_flight = 0;
    uint32_t store_phase = 0;
    auto drain_one = [&]() {   // oldest stage: wait for its load, store it to HBM, free it once the store has read it
        mbar_wait(&full[store_s], store_phase);
        bulk_s2g(dst_of[store_s], ring + (size_t)store_s * GATHER_STAGE_BYTES, GATHER_STAGE_BYTES);
        bulk_commit();
        bulk_wait_read<GATHER_PENDING>();
        if (++store_s == GATHER_STAGES) { store_s = 0; store_phase ^= 1; }
        --in_flight;
    };

    // the ids of a window are loaded one window ahead, so their latency hides behind the copies of the current one
    int32_t v[GATHER_WIN / 32], vn[GATHER_WIN / 32];
#pragma unroll
    for (int j = 0; j < GATHER_WIN / 32; ++j) {
        const int64_t t = (int64_t)j * 32 + lane;
        vn[j] = t < n_tasks ? load_id<DOOR>(ids + t) : -1;
    }
    for (int64_t base = 0; base < n_tasks; base += GATHER_WIN) {
        // ---- compact this window's valid tasks; keep the share [lo, hi) of this CTA
        int nv = 0;
#pragma unroll
        for (int j = 0; j < GATHER_WIN / 32; ++j) {
            v[j] = vn[j];
            const int64_t t = base + GATHER_WIN + j * 32 + lane;
            vn[j] = t < n_tasks ? load_id<DOOR>(ids + t) : -1;
            nv += __popc(__ballot_sync(0xffffffffu, v[j] >= 0));
        }
        const int lo = (int)((int64_t)nv * blockIdx.x / gridDim.x), hi = (int)((int64_t)nv * (blockIdx.x + 1) / gridDim.x);
        int seen = 0;
#pragma unroll
        for (int j = 0; j < GATHER_WIN / 32; ++j) {
            const unsigned b = __ballot_sync(0xffffffffu, v[j] >= 0);
            const int rank = seen + __popc(b & lt);
            if (v[j] >= 0 && rank >= lo && rank < hi) {
                q_task[rank - lo] = (int32_t)(base + j * 32 + lane);
                q_id[rank - lo] = v[j];
            }
            seen += __popc(b);
        }
        __syncwarp();
        // ---- lane 0: ring of bulk copies host -> smem -> HBM over (hi - lo) * cpb units of 16 KiB.  A stage remembers
        // its destination, so loads stay in flight across windows (no drain at a window boundary)
        if (lane == 0) {
            const int n_units = (hi - lo) * (int)cpb;
            for (int u = 0; u < n_units; ++u) {
                if (in_flight == GATHER_STAGES - GATHER_PENDING) { drain_one(); }
                const int e = u / (int)cpb, c = u % (int)cpb;
                const int64_t r = q_task[e] / topk;
                const char* src = host_kv + ((r * n_blocks + q_id[e]) * (int64_t)block_bytes + (int64_t)c * GATHER_STAGE_BYTES);
                dst_of[load_s] = pool + ((int64_t)q_task[e] * block_bytes + (int64_t)c * GATHER_STAGE_BYTES);
                mbar_arrive_expect_tx(&full[load_s], GATHER_STAGE_BYTES);
                bulk_g2s(ring + (size_t)load_s * GATHER_STAGE_BYTES, src, GATHER_STAGE_BYTES, &full[load_s]);
                if (++load_s == GATHER_STAGES) load_s = 0;
                ++in_flight;
            }
        }
        __syncwarp();   // the queue is rewritten by the next window
    }
    if (lane == 0) {
        while (in_flight > 0) drain_one();
    }
    if (lane == 0) bulk_wait<0>();  // all HBM writes complete before the kernel (and its completion event) retires
}

constexpr int LDG_UNROLL = 8;                       // 8 x 16 B in flight per lane
constexpr int LDG_UNIT_BYTES = LDG_UNROLL * 32 * 16;  // 4 KiB per warp-iteration

template <bool DOOR>
__global__ void __launch_bounds__(256) gather_ldg_kernel(const char* __restrict__ host_kv, const int32_t* ids,
                                                         char* __restrict__ pool, int n_rows, int n_blocks, int topk,
                                                         uint32_t block_bytes, unsigned int* door) {
    const int lane = threadIdx.x & 31;
    pdl_wait();
    pdl_launch_dependents();
    if (DOOR) {
        if (threadIdx.x == 0) door_wait(door, (unsigned)n_rows);
        __syncthreads();
    }
    const int64_t warp = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int64_t n_warps = (int64_t)gridDim.x * (blockDim.x >> 5);
    const uint32_t units_per_block = block_bytes / LDG_UNIT_BYTES;
    const int64_t n_units = (int64_t)n_rows * topk * units_per_block;
    for (int64_t u = warp; u < n_units; u += n_warps) {
        int64_t task = u / units_per_block;
        uint32_t c = (uint32_t)(u % units_per_block);
        int32_t id = load_id<DOOR>(ids + task);
        if (id < 0) continue;
        int64_t r = task / topk;
        const char* src = host_kv + ((r * n_blocks + id) * (int64_t)block_bytes + (int64_t)c * LDG_UNIT_BYTES) + lane * 16;
        char* dst = pool + u * (int64_t)LDG_UNIT_BYTES + lane * 16;
        int4 v[LDG_UNROLL];
#pragma unroll
        for (int i = 0; i < LDG_UNROLL; ++i) v[i] = ld_nc_v4(src + i * 512);
#pragma unroll
        for (int i = 0; i < LDG_UNROLL; ++i) st_na_v4(dst + i * 512, v[i]);
    }
}

}  // namespace

int sparda_launch_gather(sparda_ctx* ctx, const void* host_kv, int n_blocks, const int32_t* ids, int topk, void* pool,
                         cudaStream_t st) {
    const uint32_t block_bytes = 2u * ctx->cfg.block_size * ctx->cfg.head_dim * 2u;
    const int ctas = ctx->cfg.gather_ctas;
    unsigned int* door = ctx->door_next;
    if (ctx->cfg.gather_mode == SPARDA_GATHER_TMA) {
        const int smem = GATHER_STAGES * GATHER_STAGE_BYTES;
        sparda_kernel_state& ks = ctx->kstate[SPARDA_K_GATHER_TMA];
        if (!ks.attr_set) {
            SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(gather_tma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(gather_tma_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            ks.attr_set = true;
        }
        cudaLaunchAttribute at[1] = {sparda_pdl_attr()};
        cudaLaunchConfig_t lc = {};
        lc.gridDim = dim3(ctas, 1, 1);
        lc.blockDim = dim3(32, 1, 1);
        lc.dynamicSmemBytes = smem;
        lc.stream = st;
        lc.attrs = at;
        lc.numAttrs = sparda_use_pdl(ctx) ? 1 : 0;
        SPARDA_CUDA_TRY(ctx, cudaLaunchKernelEx(&lc, door ? gather_tma_kernel<true> : gather_tma_kernel<false>, (const char*)host_kv, ids, (char*)pool, ctx->R, n_blocks,
                                                topk, block_bytes, door));
    } else {
        cudaLaunchAttribute at[1] = {sparda_pdl_attr()};
        cudaLaunchConfig_t lc = {};
        lc.gridDim = dim3(ctas, 1, 1);
        lc.blockDim = dim3(256, 1, 1);
        lc.stream = st;
        lc.attrs = at;
        lc.numAttrs = sparda_use_pdl(ctx) ? 1 : 0;
        SPARDA_CUDA_TRY(ctx, cudaLaunchKernelEx(&lc, door ? gather_ldg_kernel<true> : gather_ldg_kernel<false>, (const char*)host_kv, ids, (char*)pool, ctx->R, n_blocks,
                                                topk, block_bytes, door));
    }
    SPARDA_CUDA_TRY(ctx, cudaGetLastError());
    ctx->launches++;
    return SPARDA_OK;
}
