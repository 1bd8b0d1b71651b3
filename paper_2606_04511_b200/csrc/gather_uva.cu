// Prefetch launch (a3): persistent UVA gather, pinned host memory -> HBM block pool.
//
// Alg.2 l.5, Sec.4.3: "a persistent ... kernel based on UVA ... keeps a small fixed set of
// CTAs active and lets them continuously process block-transfer tasks within a single launch".
//
// Task = one selected block (r, slot): 2*S*D*2 contiguous bytes at host_kv[(r*Nb + ids[r][slot])] ->
// dev_pool[(r*k + slot)].  ids are read from device memory when the kernel runs.
//
// Two engines, same tasks, same bytes:
//  * SPARDA_GATHER_TMA (default, B200-native): ONE thread per CTA drives a ring of 16 KiB shared-memory
//    stages with bulk-copy (TMA) instructions: cp.async.bulk global(host-mapped)->smem completing on an
//    mbarrier, then cp.async.bulk smem->global(HBM).  No registers or LSU slots are spent on payload, so a
//    handful of CTAs saturates the host link (measured on this box: 2-4 CTAs x 1 thread reach the same
//    51.4 GB/s plateau that takes 8+ CTAs x 256 threads with vector loads), leaving the SMs to the compute
//    stream (the trade-off of P:L116).
//  * SPARDA_GATHER_LDG: the paper's shape, persistent warps issuing 16-byte vector loads (8 in flight per
//    lane) from mapped host memory, 4 KiB per warp-iteration.
#include "sparda_internal.cuh"

namespace {

using namespace sparda;

constexpr int GATHER_STAGE_BYTES = 16384;
constexpr int GATHER_STAGES = 6;  // 96 KiB ring per CTA, up to 5 loads in flight while one stage drains

__global__ void __launch_bounds__(32) gather_tma_kernel(const char* __restrict__ host_kv, const int32_t* __restrict__ ids,
                                                        char* __restrict__ pool, int n_rows, int n_blocks, int topk,
                                                        uint32_t block_bytes) {
    extern __shared__ __align__(128) char ring[];
    __shared__ uint64_t full[GATHER_STAGES];
    if (threadIdx.x != 0) return;
    for (int s = 0; s < GATHER_STAGES; ++s) mbar_init(&full[s], 1);
    mbar_fence_init();
    fence_proxy_async_smem();

    const uint32_t chunks_per_block = block_bytes / GATHER_STAGE_BYTES;  // 2 at D=128, 1 at D=64
    const int64_t n_units = (int64_t)n_rows * topk * chunks_per_block;
    // unit u -> (task = u / cpb, chunk = u % cpb); static round-robin over the persistent grid
    int64_t load_u = blockIdx.x, store_u = blockIdx.x;
    int load_s = 0, store_s = 0;
    uint32_t store_phase = 0;
    int in_flight = 0;
    // a skipped (-1) unit occupies no stage: both cursors skip it identically
    auto src_of = [&](int64_t u, const char*& src) -> bool {
        int64_t task = u / chunks_per_block;
        uint32_t c = (uint32_t)(u % chunks_per_block);
        int32_t id = __ldg(ids + task);
        if (id < 0) return false;
        int64_t r = task / topk;
        src = host_kv + ((r * n_blocks + id) * (int64_t)block_bytes + (int64_t)c * GATHER_STAGE_BYTES);
        return true;
    };
    while (true) {
        // fill the ring
        while (in_flight < GATHER_STAGES && load_u < n_units) {
            const char* src;
            if (src_of(load_u, src)) {
                mbar_arrive_expect_tx(&full[load_s], GATHER_STAGE_BYTES);
                bulk_g2s(ring + (size_t)load_s * GATHER_STAGE_BYTES, src, GATHER_STAGE_BYTES, &full[load_s]);
                if (++load_s == GATHER_STAGES) load_s = 0;
                ++in_flight;
            }
            load_u += gridDim.x;
        }
        if (in_flight == 0) break;
        // drain the oldest stage
        const char* dummy;
        while (!src_of(store_u, dummy)) store_u += gridDim.x;
        mbar_wait(&full[store_s], store_phase);
        bulk_s2g(pool + store_u * (int64_t)GATHER_STAGE_BYTES, ring + (size_t)store_s * GATHER_STAGE_BYTES, GATHER_STAGE_BYTES);
        bulk_commit();
        bulk_wait_read<0>();  // the stage may be refilled once the store has read it
        if (++store_s == GATHER_STAGES) { store_s = 0; store_phase ^= 1; }
        store_u += gridDim.x;
        --in_flight;
    }
    bulk_wait<0>();  // all HBM writes complete before the kernel (and its completion event) retires
}

constexpr int LDG_UNROLL = 8;                       // 8 x 16 B in flight per lane
constexpr int LDG_UNIT_BYTES = LDG_UNROLL * 32 * 16;  // 4 KiB per warp-iteration

__global__ void __launch_bounds__(256) gather_ldg_kernel(const char* __restrict__ host_kv, const int32_t* __restrict__ ids,
                                                         char* __restrict__ pool, int n_rows, int n_blocks, int topk,
                                                         uint32_t block_bytes) {
    const int lane = threadIdx.x & 31;
    const int64_t warp = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int64_t n_warps = (int64_t)gridDim.x * (blockDim.x >> 5);
    const uint32_t units_per_block = block_bytes / LDG_UNIT_BYTES;
    const int64_t n_units = (int64_t)n_rows * topk * units_per_block;
    for (int64_t u = warp; u < n_units; u += n_warps) {
        int64_t task = u / units_per_block;
        uint32_t c = (uint32_t)(u % units_per_block);
        int32_t id = __ldg(ids + task);
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
    if (ctx->cfg.gather_mode == SPARDA_GATHER_TMA) {
        static bool attr_set = false;
        const int smem = GATHER_STAGES * GATHER_STAGE_BYTES;
        if (!attr_set) {
            SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(gather_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            attr_set = true;
        }
        gather_tma_kernel<<<ctas, 32, smem, st>>>((const char*)host_kv, ids, (char*)pool, ctx->R, n_blocks, topk, block_bytes);
    } else {
        gather_ldg_kernel<<<ctas, 256, 0, st>>>((const char*)host_kv, ids, (char*)pool, ctx->R, n_blocks, topk, block_bytes);
    }
    SPARDA_CUDA_TRY(ctx, cudaGetLastError());
    ctx->launches++;
    return SPARDA_OK;
}
