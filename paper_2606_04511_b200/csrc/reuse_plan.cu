// Step-to-step block reuse: the paper's engine keeps, per layer, the blocks selected at the previous
// decode step and fetches "only newly selected blocks" (App. C "Efficiency").  The pool of a layer therefore
// persists between steps and this kernel decides, on the device, what the prefetch has to move:
//
//   in   ids_new [R][k]   this step's selection B_l (ascending, -1 padded), as written by forecast_select
//   i/o  slot_ids[R][k]   block held by each pool slot (-1 = empty)
//   out  fetch   [R][k]   block to copy into slot s, or -1: exactly the `ids` argument of the gather kernel
//   out  n_fetch [R]      number of blocks to fetch
//
// Slot policy (reading q18): a slot whose block is selected again keeps it (no copy); the j-th smallest newly
// selected block that is not resident goes to the j-th lowest-numbered slot whose block was not selected again; slots
// left over become empty.  Attention reads the pool in slot order with slot_ids as its validity list (softmax
// attention does not depend on the order of the blocks).
//
// One warp per row: binary search of every resident block in the ascending selection, an atomicMin per hit names the
// lowest slot as its owner (so a duplicated resident block, which this kernel never produces, is still resolved as
// the oracle does), two ballot compactions list the freed slots and the missing blocks in ascending order.
#include "sparda_internal.cuh"
#include "reuse_plan.cuh"

namespace {

using namespace sparda;

constexpr int RP_WARPS = 4;

__global__ void __launch_bounds__(RP_WARPS * 32) reuse_plan_kernel(const int32_t* __restrict__ ids_new, int32_t* __restrict__ slot_ids,
                                                                    int32_t* __restrict__ fetch, int32_t* __restrict__ n_fetch,
                                                                    int n_rows, int k) {
    __shared__ ReusePlanScratch sc[RP_WARPS];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int r = blockIdx.x * RP_WARPS + w;
    if (r >= n_rows) return;
    int32_t old[RP_MAXK / 32];
    reuse_plan_load(slot_ids + (size_t)r * k, k, lane, old);
    const int n_miss = reuse_plan_row(ids_new + (size_t)r * k, slot_ids + (size_t)r * k, old, fetch + (size_t)r * k, k, sc[w], lane);
    if (lane == 0 && n_fetch) n_fetch[r] = n_miss;
}

}  // namespace
int sparda_launch_reuse_plan(sparda_ctx* ctx, const int32_t* ids_new, int topk, int32_t* slot_ids, int32_t* fetch,
                             int32_t* n_fetch, cudaStream_t st) {
    if (topk > RP_MAXK) return SPARDA_EINVAL;
    const int grid = (ctx->R + RP_WARPS - 1) / RP_WARPS;
    reuse_plan_kernel<<<grid, RP_WARPS * 32, 0, st>>>(ids_new, slot_ids, fetch, n_fetch, ctx->R, topk);
    SPARDA_CUDA_TRY(ctx, cudaGetLastError());
    ctx->launches++;
    return SPARDA_OK;
}
