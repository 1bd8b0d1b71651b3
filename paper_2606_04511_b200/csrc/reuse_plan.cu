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

namespace {

constexpr int RP_WARPS = 4;
constexpr int RP_MAXK = 256;

__global__ void __launch_bounds__(RP_WARPS * 32) reuse_plan_kernel(const int32_t* __restrict__ ids_new, int32_t* __restrict__ slot_ids,
                                                                    int32_t* __restrict__ fetch, int32_t* __restrict__ n_fetch,
                                                                    int n_rows, int k) {
    __shared__ int32_t s_new[RP_WARPS][RP_MAXK];
    __shared__ int32_t s_owner[RP_WARPS][RP_MAXK];
    __shared__ int16_t s_free[RP_WARPS][RP_MAXK], s_miss[RP_WARPS][RP_MAXK];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int r = blockIdx.x * RP_WARPS + w;
    if (r >= n_rows) return;
    const unsigned lt = (1u << lane) - 1u;
    int32_t* nw = s_new[w];
    int32_t* owner = s_owner[w];
    const int32_t* in = ids_new + (size_t)r * k;
    int32_t* slots = slot_ids + (size_t)r * k;
    int32_t* fo = fetch + (size_t)r * k;

    int m = 0;   // valid entries of the selection (ascending, then -1 padding)
    for (int c = 0; c < k; c += 32) {
        const int i = c + lane;
        const int32_t v = i < k ? in[i] : -1;
        if (i < k) { nw[i] = v; owner[i] = 0x7fffffff; }
        m += __popc(__ballot_sync(0xffffffffu, v >= 0));
    }
    __syncwarp();
    // hits: resident blocks that are selected again
    for (int c = 0; c < k; c += 32) {
        const int s = c + lane;
        const int32_t b = s < k ? slots[s] : -1;
        if (b >= 0) {
            int lo = 0, hi = m;
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (nw[mid] < b) lo = mid + 1; else hi = mid;
            }
            if (lo < m && nw[lo] == b) atomicMin(&owner[lo], s);
        }
    }
    __syncwarp();
    // freed slots (ascending) and missing blocks (ascending position = ascending id)
    int n_free = 0, n_miss = 0;
    for (int c = 0; c < k; c += 32) {
        const int s = c + lane;
        bool kept = false;
        if (s < k) {
            const int32_t b = slots[s];
            if (b >= 0) {
                int lo = 0, hi = m;
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (nw[mid] < b) lo = mid + 1; else hi = mid;
                }
                kept = lo < m && nw[lo] == b && owner[lo] == s;
            }
        }
        const unsigned fb = __ballot_sync(0xffffffffu, s < k && !kept);
        if (s < k && !kept) s_free[w][n_free + __popc(fb & lt)] = (int16_t)s;
        n_free += __popc(fb);
        const bool miss = s < m && owner[s] == 0x7fffffff;
        const unsigned mb = __ballot_sync(0xffffffffu, miss);
        if (miss) s_miss[w][n_miss + __popc(mb & lt)] = (int16_t)s;
        n_miss += __popc(mb);
        if (s < k && kept) fo[s] = -1;
    }
    __syncwarp();
    for (int j = lane; j < n_free; j += 32) {
        const int s = s_free[w][j];
        const int32_t b = j < n_miss ? nw[s_miss[w][j]] : -1;
        slots[s] = b;
        fo[s] = b;
    }
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
