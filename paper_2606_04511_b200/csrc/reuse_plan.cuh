// One row of the step-to-step block-reuse plan (f1; slot policy = reading q18), executed by one warp.  Shared by
// reuse_plan_kernel (reuse_plan.cu) and the fused tail of forecast_select_kernel (select_decode.cu).
#pragma once
#include <stdint.h>

namespace sparda {

constexpr int RP_MAXK = 256;

struct ReusePlanScratch {   // per warp, shared memory
    int32_t nw[RP_MAXK];
    int32_t owner[RP_MAXK];
    int16_t sfree[RP_MAXK], smiss[RP_MAXK];
};

// in [k]: this step's selection (ascending, -1 padded); slots [k] in/out; fo [k] out.  Returns the number of fetches.
// in == nullptr: the selection is already in sc.nw (written by the selecting CTA as it emitted the ids: the fused tail of
// forecast_select_kernel, which thereby skips a round trip through L2).
// The row's slot table is passed in registers (lane l holds slots[32 q + l] in old[q]): reuse_plan_load() reads it, and a
// caller with something else to do first issues that read early.
__device__ __forceinline__ void reuse_plan_load(const int32_t* slots, int k, int lane, int32_t (&old)[RP_MAXK / 32]) {
#pragma unroll
    for (int q = 0; q < RP_MAXK / 32; ++q) old[q] = q * 32 + lane < k ? slots[q * 32 + lane] : -1;
}

__device__ __forceinline__ int reuse_plan_row(const int32_t* in, int32_t* slots, const int32_t (&old)[RP_MAXK / 32], int32_t* fo, int k,
                                              ReusePlanScratch& sc, int lane) {
    int32_t* nw = sc.nw;
    int32_t* owner = sc.owner;
    int16_t* sfree = sc.sfree;
    int16_t* smiss = sc.smiss;
    const unsigned lt = (1u << lane) - 1u;

    int m = 0;   // valid entries of the selection (ascending, then -1 padding)
    for (int c = 0; c < k; c += 32) {
        const int i = c + lane;
        const int32_t v = i < k ? (in ? __ldcg(in + i) : nw[i]) : -1;
        if (i < k) { nw[i] = v; owner[i] = 0x7fffffff; }
        m += __popc(__ballot_sync(0xffffffffu, v >= 0));
    }
    __syncwarp();

    // hits: resident blocks that are selected again (hit[q] = position of slot 32 q + lane's block in the selection, or -1)
    int hit[RP_MAXK / 32];
#pragma unroll
    for (int q = 0; q < RP_MAXK / 32; ++q) {
        const int c = q * 32;
        hit[q] = -1;
        if (c >= k) break;
        const int s = c + lane;
        const int32_t b = old[q];
        if (b >= 0) {
            int lo = 0, hi = m;
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (nw[mid] < b) lo = mid + 1; else hi = mid;
            }
            if (lo < m && nw[lo] == b) { hit[q] = lo; atomicMin(&owner[lo], s); }
        }
    }
    __syncwarp();
    // freed slots (ascending) and missing blocks (ascending position = ascending id)
    int n_free = 0, n_miss = 0;
#pragma unroll
    for (int q = 0; q < RP_MAXK / 32; ++q) {
        const int c = q * 32;
        if (c >= k) break;
        const int s = c + lane;
        const bool kept = s < k && hit[q] >= 0 && owner[hit[q]] == s;   // the lowest slot holding the block keeps it
        const unsigned fb = __ballot_sync(0xffffffffu, s < k && !kept);
        if (s < k && !kept) sfree[n_free + __popc(fb & lt)] = (int16_t)s;
        n_free += __popc(fb);
        const bool miss = s < m && owner[s] == 0x7fffffff;
        const unsigned mb = __ballot_sync(0xffffffffu, miss);
        if (miss) smiss[n_miss + __popc(mb & lt)] = (int16_t)s;
        n_miss += __popc(mb);
        if (s < k && kept) fo[s] = -1;
    }
    __syncwarp();
    for (int j = lane; j < n_free; j += 32) {
        const int s = sfree[j];
        const int32_t b = j < n_miss ? nw[smiss[j]] : -1;
        slots[s] = b;
        fo[s] = b;
    }
    return n_miss;
}

}  // namespace sparda
