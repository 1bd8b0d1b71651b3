// Forecast indexer for decode (a1 + a2) and key compression (a0).
//
//   s[r,j] = sum_d F[r,d] * Kpool[r,j,d]      Eq.4: raw logits, no softmax, no scale
//   ids[r] = f_top(s[r, 0:n_cand], k)          P:L78: k best blocks, ties -> lowest id, ascending ids, -1 padded
//
// One launch, one thread-block cluster per row r.  The row's n_cand pooled keys are cut into CS contiguous ranges,
// one per CTA of the cluster (CS = 1..16, chosen so that R*CS covers every SM, up to two CTAs per SM).  In every CTA a
// producer thread streams its range through a ring of 16 KiB shared-memory stages with TMA tensor-map loads (64-key x
// 64-element boxes, 128-byte swizzle, completing on mbarriers: 96 KiB in flight per CTA, no registers or LSU slots spent
// on the stream).  HBM-bound (R*n_cand*D*2 bytes of Kpool, 1 FLOP per byte), so the arithmetic must cost next to
// nothing in issue slots: the 8 consumer warps read the swizzled stage with conflict-free ldmatrix and take the dot
// products with mma.sync.m16n8k16 (16 keys as the M rows, F in column 0 of the B operand, fp32 accumulate): 8 ldmatrix +
// 8 mma per 16 keys instead of ~160 warp instructions of convert + FMA + shuffle, which had 8 warps per SM running at the
// HBM rate with nothing to spare (sm__warps_active 14 %, round 1).  The tensor pipe is not what this is for (7 of its 8
// output columns are zero); the point is the issue slots.  Order-preserving uint32 keys go straight into the shared
// memory of the cluster's CTA 0 (DSMEM), min / max by red.shared::cluster.  After one cluster barrier CTA 0 holds the
// whole row's scores on chip and selects: a one-pass 256-bucket value histogram finds the boundary bucket of the k-th
// largest, every warp ranks its few members exactly, and an index-ordered compaction emits {key > T} plus the first
// (k - #{key > T}) keys == T, which is exactly "sort by (score desc, id asc), take k, sort by id".  Scores never touch
// global memory; there is no ticket, no fence and no scratch.
//
// Debug builds only (-DSPARDA_TRACE, never shipped): per-CTA globaltimer stamps of the phases, read back by a probe
// through sparda_debug_set_sel_trace.
#include "sparda_internal.cuh"
#include "reuse_plan.cuh"

#ifdef SPARDA_TRACE
// per-CTA timeline: thread 0 stamps the SM cycle counter at up to 16 points (relative to kernel entry) and appends
// (blockIdx, globaltimer at entry, globaltimer at exit, cycles[16]) to a log when it leaves
__device__ unsigned long long* g_sel_log;      // [0] = cursor, then 20 words per entry from word 8
extern "C" void sparda_debug_set_sel_log(unsigned long long* p) { cudaMemcpyToSymbol(g_sel_log, &p, sizeof(p)); }
__device__ __forceinline__ unsigned long long sel_now() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
struct SelCyc { unsigned long long t0; long long c0; long long c[16]; };
#define SEL_LOG_DECL SelCyc cyc_; cyc_.t0 = sel_now(); cyc_.c0 = clock64(); _Pragma("unroll") for (int i_ = 0; i_ < 16; ++i_) cyc_.c[i_] = 0; \
    __shared__ long long s_dbg[4];
#define SEL_CYC(i) if (threadIdx.x == 0) cyc_.c[i] = clock64() - cyc_.c0;
#define SEL_CYC_PRODUCER(i) s_dbg[i] = clock64();
#define SEL_LOG_EXIT                                                                          \
    if (threadIdx.x == 0 && g_sel_log) {                                                      \
        cyc_.c[14] = s_dbg[0] - cyc_.c0; cyc_.c[15] = s_dbg[1] - cyc_.c0;                     \
        unsigned long long e_ = atomicAdd(g_sel_log, 1ull);                                   \
        unsigned long long* d_ = g_sel_log + 8 + e_ * 20;                                     \
        d_[0] = blockIdx.x; d_[1] = cyc_.t0; d_[2] = sel_now(); d_[3] = (unsigned long long)(clock64() - cyc_.c0); \
        _Pragma("unroll") for (int i_ = 0; i_ < 16; ++i_) d_[4 + i_] = (unsigned long long)cyc_.c[i_];           \
    }
#else
struct SelCyc {};
#define SEL_LOG_DECL SelCyc cyc_;
#define SEL_CYC(i)
#define SEL_CYC_PRODUCER(i)
#define SEL_LOG_EXIT
#endif

namespace {

using namespace sparda;

constexpr int SEL_THREADS = 256;                  // consumer threads (the selection runs on these)
constexpr int SEL_CTA_THREADS = SEL_THREADS + 32; // + one producer warp
constexpr int SEL_STAGE_BYTES = 16384;            // two 64 x 64-element TMA boxes
constexpr int SEL_STAGES = 6;

// barrier of the 256 consumer threads only (the producer warp has left by the time the selection runs)
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive1(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// address of `local` in the shared memory of CTA `rank` of this cluster (shared::cluster window)
__device__ __forceinline__ uint32_t map_to_cta(const void* local, uint32_t rank) {
    uint32_t out;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(out) : "r"(smem_u32(local)), "r"(rank));
    return out;
}
// asynchronous store into the shared memory of a CTA of the cluster that also counts its bytes on an mbarrier there
// (st.async ... complete_tx): the receiver waits for "all bytes have landed", the sender never waits for its stores
__device__ __forceinline__ void st_async_u32(uint32_t addr, uint32_t v, uint32_t mbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.u32 [%0], %1, [%2];" ::"r"(addr), "r"(v), "r"(mbar) : "memory");
}
__device__ __forceinline__ void st_async_v2_u32(uint32_t addr, uint32_t a, uint32_t b, uint32_t mbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.u32 [%0], {%1, %2}, [%3];" ::"r"(addr), "r"(a), "r"(b), "r"(mbar)
                 : "memory");
}

__device__ __forceinline__ uint32_t block_incl_scan_256(uint32_t v, uint32_t* warp_tot /*[8]*/, uint32_t& total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t n = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += n;
    }
    if (lane == 31) warp_tot[w] = v;
    consumer_sync();
    uint32_t add = 0, tot = 0;
#pragma unroll
    for (int i = 0; i < SEL_THREADS / 32; ++i) {
        uint32_t t = warp_tot[i];
        if (i < w) add += t;
        tot += t;
    }
    total = tot;
    consumer_sync();
    return v + add;
}

__device__ __forceinline__ float key_to_float(uint32_t key) {
    // inverse of orderable(): positive floats carry the top bit (flip it back), negative ones are complemented
    return __uint_as_float(key ^ (~(uint32_t)((int32_t)key >> 31) | 0x80000000u));
}

constexpr int SEL_CAND_CAP = 32;  // boundary-bucket size the exact finish handles

// Exact top-k over keys[0..n) (order-preserving uint32 keys in shared memory), k < n <= 8192.  256 consumer threads.
//
// The tail of the kernel is a chain of dependent instructions on 8 warps, so it is written for few instructions and two
// CTA barriers (round 1: 5600 cycles with three barriers and a generic-address key array; this version: see DESIGN.md 5.1):
//  1. every thread loads its contiguous slice (16-byte loads; the first 8 keys and their buckets stay in registers) and
//     counts it into 256 equal-width value buckets of the row's [min, max].  The bucket map is monotone (one FMA with a
//     positive scale, clamp, truncate), so every key in a higher bucket is larger than every key in a lower one and
//     equal keys share a bucket.  Only the upper 128 buckets are counted at first: the k-th largest of n >> k keys lies
//     above the middle of the range unless the row has a far positive outlier, and shared-memory atomics (bank
//     conflicts) are what this pass costs; if the upper half holds fewer than k keys a second round counts the lower.
//  2. every warp redundantly suffix-scans 128 counts (4 per lane + one shuffle scan) and finds the boundary bucket b*
//     of the k-th largest -- no broadcast.  A thread marks its keys above b* in a register bit mask, the members of b*
//     (<= 32, typically ~4) go to a list; the strict counts are scanned per warp BEFORE the second barrier.
//  3. every warp redundantly ranks the list by (key desc, id asc) with shuffles: member f is taken iff its rank is below
//     need = k - #{key above b*}; a thread's output position is (warps before) + (lanes before) + (taken members with
//     a smaller index), and ids are emitted in index order: exactly "sort by (score desc, id asc), take k, sort by id".
// Fallback (heavy ties / degenerate range): exact MSB-first 8-bit radix select + index-ordered compaction.
__device__ __forceinline__ void topk_emit(const uint32_t* keys, int n, int k, uint32_t kmin, uint32_t kmax, int32_t* ids_out,
                          int32_t* ids_smem /* optional copy of the row's ids for the fused reuse plan, or nullptr */,
                          uint32_t* hist /*[256], zeroed*/, uint32_t* warp_tot /*[8]*/, uint32_t* bcast /*[4], [2] zeroed*/,
                          uint32_t* cand /*[2 * SEL_CAND_CAP]*/, SelCyc& cyc_) {
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    // a thread's contiguous slice: a multiple of 4 keys (16-byte loads), <= 32 so that it fits one bit mask
    const int per = (((n + SEL_THREADS - 1) / SEL_THREADS) + 3) & ~3;
    const int lo = min(tid * per, n), hi = min(lo + per, n);
    const float flo = key_to_float(kmin), fhi = key_to_float(kmax);
    const float scale = __fdividef(256.0f, fhi - flo), shift = -flo * scale;   // any positive scale keeps the map monotone
    bool fast = (kmax > kmin) && (scale > 0.f) && (scale < INFINITY) && (fabsf(shift) < INFINITY);
    auto bucket = [&](uint32_t key) -> int {   // monotone in key; NaN (forced keys of the grid mode) -> 255
        return (int)fminf(fmaf(key_to_float(key), scale, shift), 255.0f);
    };
    if (fast) {
        SEL_CYC(6);
        // ---- 1. buckets of the slice; count the upper half
        int bk[8];
        {
            uint32_t kr[8];
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const uint4 v = lo + 4 * q < hi ? *reinterpret_cast<const uint4*>(keys + lo + 4 * q) : make_uint4(0, 0, 0, 0);
                kr[4 * q] = v.x; kr[4 * q + 1] = v.y; kr[4 * q + 2] = v.z; kr[4 * q + 3] = v.w;
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) bk[j] = lo + j < hi ? bucket(kr[j]) : -1;
#pragma unroll
            for (int j = 0; j < 8; ++j)
                if (bk[j] >= 128) atomicAdd(&hist[bk[j]], 1u);
            for (int i = lo + 8; i < hi; ++i) {   // n > 2048 only
                const int b = bucket(keys[i]);
                if (b >= 128) atomicAdd(&hist[b], 1u);
            }
        }
        consumer_sync();
        SEL_CYC(7);
        // ---- 2. boundary bucket: suffix counts of 128 buckets, redundantly per warp (lane l owns buckets top - 4l - j)
        int bstar = -1;
        uint32_t need = 0, pop = 0, above = 0;
#pragma unroll 1
        for (int top = 255; top >= 127; top -= 128) {
            const uint4 hv = *reinterpret_cast<const uint4*>(hist + top - 3 - 4 * lane);
            const uint32_t h[4] = {hv.w, hv.z, hv.y, hv.x};   // descending bucket
            const uint32_t run = h[0] + h[1] + h[2] + h[3];
            uint32_t incl = run;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t nb = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += nb;
            }
            uint32_t gt = above + incl - run;                     // keys in buckets above this lane's four
            int my_b = -1;
            uint32_t my_need = 0, my_pop = 0;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (gt < (uint32_t)k && (uint32_t)k <= gt + h[j]) { my_b = top - 4 * lane - j; my_need = k - gt; my_pop = h[j]; }
                gt += h[j];
            }
            const unsigned found = __ballot_sync(0xffffffffu, my_b >= 0);
            if (found) {
                const int src = __ffs(found) - 1;
                bstar = __shfl_sync(0xffffffffu, my_b, src);
                need = __shfl_sync(0xffffffffu, my_need, src);
                pop = __shfl_sync(0xffffffffu, my_pop, src);
                break;
            }
            // fewer than k keys in the upper half (a far positive outlier stretches the range): count the lower half too
            above = __shfl_sync(0xffffffffu, above + incl, 31);
#pragma unroll
            for (int j = 0; j < 8; ++j)
                if (bk[j] >= 0 && bk[j] < 128) atomicAdd(&hist[bk[j]], 1u);
            for (int i = lo + 8; i < hi; ++i) {
                const int b = bucket(keys[i]);
                if (b < 128) atomicAdd(&hist[b], 1u);
            }
            consumer_sync();
        }
        SEL_CYC(8);
        if (bstar >= 0 && pop <= SEL_CAND_CAP) {
            // ---- mark; strict counts scanned per warp before the barrier
            uint32_t m_sel = 0, m_eq = 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                if (bk[j] > bstar) m_sel |= 1u << j;
                if (bk[j] == bstar) m_eq |= 1u << j;
            }
            for (int i = lo + 8; i < hi; ++i) {
                const int b = bucket(keys[i]);
                if (b > bstar) m_sel |= 1u << (i - lo);
                if (b == bstar) m_eq |= 1u << (i - lo);
            }
            if (m_eq) {   // few threads: one reservation per thread, then plain stores
                uint32_t s = atomicAdd(&bcast[2], (uint32_t)__popc(m_eq));
                for (uint32_t m = m_eq; m; m &= m - 1) {
                    const int j = __ffs(m) - 1;
                    cand[2 * s] = keys[lo + j];
                    cand[2 * s + 1] = (uint32_t)(lo + j);
                    ++s;
                }
            }
            const uint32_t c_strict = __popc(m_sel);
            uint32_t inc = c_strict;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t nb = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += nb;
            }
            if (lane == 31) warp_tot[w] = inc;
            consumer_sync();
        SEL_CYC(9);
            // ---- 3. rank the boundary bucket, redundantly per warp: lane f holds member f; taken iff rank < need
            const bool have = (uint32_t)lane < pop;
            const uint32_t mk = have ? cand[2 * lane] : 0u, mi = have ? cand[2 * lane + 1] : 0xFFFFFFFFu;
            uint32_t rank = 0;
            for (uint32_t f = 0; f < pop; ++f) {
                const uint32_t fk = __shfl_sync(0xffffffffu, mk, f), fi = __shfl_sync(0xffffffffu, mi, f);
                rank += (fk > mk || (fk == mk && fi < mi)) ? 1u : 0u;
            }
            const uint32_t tagged = (have && rank < need) ? mi : 0xFFFFFFFFu;   // index of a taken member, else "none"
        SEL_CYC(10);
            // position = strict keys before this thread + taken members with a smaller index; own taken members join the mask
            uint32_t pos = inc - c_strict;
            {
                const uint4 wa = *reinterpret_cast<const uint4*>(warp_tot), wb = *reinterpret_cast<const uint4*>(warp_tot + 4);
                const uint32_t wt[8] = {wa.x, wa.y, wa.z, wa.w, wb.x, wb.y, wb.z, wb.w};
#pragma unroll
                for (int i = 0; i < SEL_THREADS / 32; ++i) pos += i < w ? wt[i] : 0u;
            }
            for (uint32_t f = 0; f < pop; ++f) {
                const uint32_t ti = __shfl_sync(0xffffffffu, tagged, f);
                if (ti < (uint32_t)lo) ++pos;
                else if (ti < (uint32_t)hi) m_sel |= 1u << (ti - lo);
            }
        SEL_CYC(11);
            while (m_sel) {
                const int j = __ffs(m_sel) - 1;
                m_sel &= m_sel - 1;
                if (ids_smem) ids_smem[pos] = lo + j;
                ids_out[pos++] = lo + j;
            }
            return;
        }
        consumer_sync();   // the fallback reuses hist
    }
    // ---- fallback: exact radix select of the k-th largest key T, then take every key > T and the first krem keys == T
    uint32_t T = 0, krem = (uint32_t)k;
    {
        uint32_t prefix = 0, mask = 0;
#pragma unroll 1
        for (int shift = 24; shift >= 0; shift -= 8) {
            hist[tid] = 0;
            consumer_sync();
            for (int i = tid; i < n; i += SEL_THREADS) {
                uint32_t key = keys[i];
                if ((key & mask) == prefix) atomicAdd(&hist[(key >> shift) & 255u], 1u);
            }
            consumer_sync();
            uint32_t mine = hist[255 - tid], tot;
            uint32_t ge = block_incl_scan_256(mine, warp_tot, tot);
            uint32_t gt = ge - mine;
            if (gt < krem && krem <= ge) {
                bcast[0] = prefix | ((uint32_t)(255 - tid) << shift);
                bcast[1] = krem - gt;
            }
            consumer_sync();
            prefix = bcast[0];
            krem = bcast[1];
            mask |= 0xFFu << shift;
            consumer_sync();
        }
        T = prefix;
    }
    uint32_t c = 0;  // low 16 bits: #gt, high 16 bits: #eq  (n <= 8192)
    for (int i = lo; i < hi; ++i) {
        uint32_t key = keys[i];
        c += (key > T ? 1u : 0u) + (key == T ? 0x10000u : 0u);
    }
    uint32_t tot;
    uint32_t incl = block_incl_scan_256(c, warp_tot, tot);
    uint32_t excl = incl - c;
    uint32_t gt_before = excl & 0xFFFFu, eq_before = excl >> 16;
    uint32_t pos = gt_before + min(eq_before, krem);
    for (int i = lo; i < hi; ++i) {
        uint32_t key = keys[i];
        if (key > T) {
            if (ids_smem) ids_smem[pos] = i;
            ids_out[pos++] = i;
        } else if (key == T) {
            if (eq_before < krem) {
                if (ids_smem) ids_smem[pos] = i;
                ids_out[pos++] = i;
            }
            ++eq_before;
        }
    }
}


struct SelParams {
    const uint32_t* F;   // [R][D] bf16 pairs
    int32_t* ids;
    int n_blocks, n_cand, topk;
    int per;   // candidates (blocks) per CTA of the cluster (the last CTA's range may be shorter or empty)
    // grid mode (f3): Kpool is the (32,16) compressed-key grid, 4 keys per block; keys_valid = 4*n_cand - 1 of them exist;
    // blocks [0, n_init) and [n_cand - n_local, n_cand) are always selected
    int keys_valid, n_init, n_local;
    // optional fused reuse plan (f1, reuse_plan.cuh): after the row's ids are out, one warp of the selecting CTA updates
    // the row's slot table and fetch list -- one launch less per layer of the cached decode step
    int32_t* slot_ids;
    int32_t* fetch;
    int32_t* n_fetch;
    // optional doorbell (overlapped decode step): the CTA that owns the row rings it once the row's ids (and fetch list) are
    // out, so the gather of the layer -- already resident on its own stream -- starts without a kernel boundary in between
    unsigned int* door;
};

// tmap: the pooled keys as a [R * n_blocks * KPB][D] bf16 tensor, box = 64 keys x 64 elements, 128-byte swizzle.
template <int D, bool GRID>
__global__ void __launch_bounds__(SEL_CTA_THREADS, 2) forecast_select_kernel(const __grid_constant__ CUtensorMap tmap, SelParams p) {
    constexpr int KPB = GRID ? 4 : 1;                // keys per candidate block
    constexpr int NW = SEL_THREADS / 32;
    constexpr int ROW_BYTES = D * 2;
    constexpr int KPS = SEL_STAGE_BYTES / ROW_BYTES; // keys per stage: 64 (D = 128) or 128 (D = 64)
    constexpr int TPW = KPS / 64;                    // 16-key MMA tiles per warp per stage (4 warps share a stage)
    constexpr int KSTEPS = D / 16;                   // k-steps of the contraction
    SEL_LOG_DECL
    extern __shared__ uint8_t sel_smem_raw[];
    __shared__ uint64_t s_full[SEL_STAGES], s_empty[SEL_STAGES];
    __shared__ uint64_t s_done;                      // CTA 0: completes when every key and every warp's min / max has landed (tx bytes)
    __shared__ __align__(16) uint32_t s_hist[256];
    __shared__ __align__(16) uint32_t s_wtot[8];
    __shared__ uint32_t s_bcast[4];
    __shared__ uint32_t s_cand[2 * SEL_CAND_CAP];
    __shared__ __align__(8) uint32_t s_mm[16 * NW][2];   // per (CTA of the cluster, warp): min / max key; lives in CTA 0
    __shared__ ReusePlanScratch s_plan;

    // swizzle atoms are 1 KiB; the offset is taken in the shared window so that ring / s_keys stay shared-space pointers
    uint8_t* ring = sel_smem_raw + ((1024u - (smem_u32(sel_smem_raw) & 1023u)) & 1023u);
    uint32_t* s_keys = reinterpret_cast<uint32_t*>(ring + SEL_STAGES * SEL_STAGE_BYTES);   // [n_cand], used in CTA 0

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const uint32_t c = cluster_ctarank();
    uint32_t CS;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(CS));
    const int r = blockIdx.x / CS;
    int32_t* ids_row = p.ids + (size_t)r * p.topk;

    if (p.n_cand <= p.topk) {  // every candidate is selected (reading q5); no scoring needed
        pdl_wait();
        pdl_launch_dependents();
        if (c == 0) {
            for (int i = tid; i < p.topk; i += SEL_CTA_THREADS) ids_row[i] = i < p.n_cand ? i : -1;
            if (p.slot_ids) {
                __syncthreads();
                if (w == 0) {
                    int32_t old[RP_MAXK / 32];
                    reuse_plan_load(p.slot_ids + (size_t)r * p.topk, p.topk, lane, old);
                    const int nm = reuse_plan_row(ids_row, p.slot_ids + (size_t)r * p.topk, old, p.fetch + (size_t)r * p.topk, p.topk, s_plan, lane);
                    if (lane == 0 && p.n_fetch) p.n_fetch[r] = nm;
                }
            }
            if (p.door) {
                __syncthreads();
                if (tid == 0) door_ring(p.door);
            }
        }
        return;
    }

    const int k_lo = min((int)c * p.per, p.n_cand);
    const int n_local = min(p.per, p.n_cand - k_lo);
    const int n_keys_local = n_local * KPB;         // rows of Kpool this CTA streams
    const int n_st = (n_keys_local + KPS - 1) / KPS;
    const int row0 = (r * p.n_blocks + k_lo) * KPB; // first row of this CTA's range in the tensor map

    // one stage = up to two boxes: D = 128: the two 64-element halves of 64 keys; D = 64: two groups of 64 keys
    auto issue_stage = [&](int i) {
        const int s = i % SEL_STAGES;
        const int nk = min(KPS, n_keys_local - i * KPS);
        const int nbox = (D == 64 && nk <= 64) ? 1 : 2;
        uint8_t* dst = ring + (size_t)s * SEL_STAGE_BYTES;
        mbar_arrive_expect_tx(&s_full[s], (uint32_t)nbox * 8192u);
        tma_load_2d(dst, &tmap, 0, row0 + i * KPS, &s_full[s]);
        if (nbox == 2) tma_load_2d(dst + 8192, &tmap, D == 128 ? 64 : 0, row0 + i * KPS + (D == 128 ? 0 : 64), &s_full[s]);
    };

    SEL_CYC(0);
    if (w == NW && lane == 0) {   // the producer thread arms the barriers
        for (int s = 0; s < SEL_STAGES; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], NW / 2); }
        mbar_init(&s_done, 1);
        // CTA 0 expects one 4-byte key per candidate and one (min, max) pair per consumer warp of the cluster
        if (c == 0) mbar_arrive_expect_tx(&s_done, (uint32_t)p.n_cand * 4u + CS * NW * 8u);
        mbar_fence_init();
        fence_proxy_async_smem();
        tma_prefetch_desc(&tmap);
        SEL_CYC_PRODUCER(0);
    }
    if (tid < 256) s_hist[tid] = 0;
    if (tid == 0) s_bcast[2] = 0;
    __syncthreads();
    // All CTAs of the cluster must be running before anyone touches a neighbour's shared memory: arrive now, wait just
    // before the first remote store (by then every CTA has long arrived: the wait is free).  The release / acquire pair
    // also orders CTA 0's initialisation of s_done before the first remote store that counts on it.
    cluster_arrive();
    // Programmatic dependent launch: everything above overlaps the previous kernel's tail, and so does the producer's
    // stream of pooled keys below -- the ring fills (96 KiB per CTA) while the predecessor drains.  That is safe because a
    // dependent only starts early behind a kernel that signals launch completion early, and the kernels of this library
    // that do (select, gather, attention, projection) never write pooled keys; behind any other kernel (pool_keys,
    // append_kv, a caller's own) this launch starts after that kernel has completed (include/sparda.h, cfg.no_pdl).
    // Everything the predecessor may have written -- F, the slot table -- and every store waits for it (consumers).
    if (w != NW) {
        pdl_wait();
        pdl_launch_dependents();
    }
    SEL_CYC(1);
    // fused reuse plan: the row's slot table is needed only after the selection; its load is issued now (warp 0 of CTA 0)
    int32_t plan_old[RP_MAXK / 32];
    if (p.slot_ids && c == 0 && w == 0) reuse_plan_load(p.slot_ids + (size_t)r * p.topk, p.topk, lane, plan_old);

    if (w == NW) {
        // =============================== producer warp: the stream ===============================
        // (measured: loads issued BEFORE the CTA barrier and the cluster arrive above land 2400 cycles later than loads
        // issued here -- the async unit does not start a shared::cluster copy until the cluster is up)
        if (lane == 0) {
            for (int i = 0; i < n_st; ++i) {
                if (i >= SEL_STAGES) mbar_wait(&s_empty[i % SEL_STAGES], ((i / SEL_STAGES) - 1) & 1);
                issue_stage(i);
                if (i == SEL_STAGES - 1 || i == n_st - 1) { SEL_CYC_PRODUCER(1); }
            }
        }
        __syncwarp();
        cluster_wait();
    } else {
        // =============================== consumers: a1, scores of this CTA's range ===============================
        // Warps 0-3 take the even stages, warps 4-7 the odd ones; inside a stage warp wi owns the 16-key tiles wi, wi + 4.
        const int grp = w >> 2, wi = w & 3;
        const int gid = lane >> 2, tig = lane & 3;
        // B operand: F in column 0 (rows k of the 16 x 8 tile), zeros elsewhere: only the lanes with gid == 0 hold data
        uint32_t fb[KSTEPS][2];
        {
            const uint32_t* frow = p.F + (size_t)r * (D / 2);
#pragma unroll
            for (int ks = 0; ks < KSTEPS; ++ks) {
                fb[ks][0] = gid == 0 ? __ldg(frow + ks * 8 + tig) : 0u;
                fb[ks][1] = gid == 0 ? __ldg(frow + ks * 8 + 4 + tig) : 0u;
            }
        }
        const uint32_t keys0 = map_to_cta(s_keys, 0);          // the row's key array lives in CTA 0
        const uint32_t done0 = map_to_cta(&s_done, 0);         // ... and so does the barrier that counts what has landed
        const int mi = lane >> 3, ri = lane & 7;                // ldmatrix: this lane addresses row ri of matrix mi
        uint32_t kmin = 0xFFFFFFFFu, kmax = 0u;
        bool waited = false;
        for (int i = grp; i < n_st; i += 2) {
            const int s = i % SEL_STAGES;
            const int nk = min(KPS, n_keys_local - i * KPS);
            mbar_wait(&s_full[s], (i / SEL_STAGES) & 1);
            if (i == 0) { SEL_CYC(2); }
            const uint32_t st = smem_u32(ring + (size_t)s * SEL_STAGE_BYTES);
            // A operand: 16 keys x 16 elements per ldmatrix.x4 (matrices: rows 0-7 / 8-15 x element halves), swizzled rows
            uint32_t a[TPW][KSTEPS][4];
#pragma unroll
            for (int t = 0; t < TPW; ++t) {
                const int krow = (wi + 4 * t) * 16 + (mi & 1) * 8 + ri;                       // key within the stage
                const uint32_t rowaddr = st + (D == 64 ? (krow >> 6) * 8192 : 0) + (krow & 63) * 128;
#pragma unroll
                for (int ks = 0; ks < KSTEPS; ++ks) {
                    const int ch = ks * 2 + (mi >> 1);                                        // 16-byte chunk of the key row
                    ldmatrix_x4(rowaddr + (ch >> 3) * 8192 + (((ch & 7) ^ ri) << 4), a[t][ks][0], a[t][ks][1], a[t][ks][2], a[t][ks][3]);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive1(&s_empty[s]);            // the stage is in registers: hand it back
            if (!waited) { cluster_wait(); waited = true; }
#pragma unroll
            for (int t = 0; t < TPW; ++t) {
                float acc0[4] = {0.f, 0.f, 0.f, 0.f}, acc1[4] = {0.f, 0.f, 0.f, 0.f};   // two chains: half the dependent latency
#pragma unroll
                for (int ks = 0; ks < KSTEPS; ks += 2) {
                    mma_bf16_16816(acc0, a[t][ks], fb[ks][0], fb[ks][1]);
                    mma_bf16_16816(acc1, a[t][ks + 1], fb[ks + 1][0], fb[ks + 1][1]);
                }
                // column 0 of the 16 x 8 result: lanes with tig == 0 hold key gid (c0) and key gid + 8 (c2)
                const float sc[2] = {acc0[0] + acc1[0], acc0[2] + acc1[2]};
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int kl = (wi + 4 * t) * 16 + h * 8 + gid;                           // key within the stage
                    if (GRID) {
                        // f_top's max-pool (reading q19): block score = max over the compressed keys that start in
                        // the block = keys 4b .. 4b+3 = four consecutive gid
                        const int jkey = (k_lo * 4 + i * KPS) + kl;                           // compressed key index in the row
                        float bsc = jkey < p.keys_valid ? sc[h] : -INFINITY;
                        bsc = fmaxf(bsc, __shfl_xor_sync(0xffffffffu, bsc, 4));
                        bsc = fmaxf(bsc, __shfl_xor_sync(0xffffffffu, bsc, 8));
                        const int blk = i * (KPS / 4) + (kl >> 2);                            // block within this CTA's range
                        if (tig == 0 && (gid & 3) == 0 && blk < n_local) {
                            const int b = k_lo + blk;
                            const bool forced = b < p.n_init || b >= p.n_cand - p.n_local;   // init / local blocks: always attended
                            const uint32_t key = forced ? 0xFFFFFFFFu : orderable(bsc + 0.0f);
                            st_async_u32(keys0 + 4u * (uint32_t)b, key, done0);
                            if (!forced) { kmin = min(kmin, key); kmax = max(kmax, key); }
                        }
                    } else if (tig == 0 && kl < nk) {
                        const uint32_t key = orderable(sc[h] + 0.0f);      // +0: -0 -> +0
                        st_async_u32(keys0 + 4u * (uint32_t)(k_lo + i * KPS + kl), key, done0);
                        kmin = min(kmin, key);
                        kmax = max(kmax, key);
                    }
                }
            }
        }
        SEL_CYC(3);
        if (!waited) cluster_wait();
        kmin = __reduce_min_sync(0xffffffffu, kmin);
        kmax = __reduce_max_sync(0xffffffffu, kmax);
        // the keys went out as asynchronous stores that count their bytes on CTA 0's barrier; so does this warp's (min, max):
        // no release, no drain -- the sender is done, and CTAs 1.. leave at once (nobody reads their shared memory)
        if (lane == 0) st_async_v2_u32(map_to_cta(&s_mm[c * NW + w][0], 0), kmin, kmax, done0);
    }
    SEL_CYC(4);
    if (c != 0 || w == NW) { SEL_LOG_EXIT return; }
    mbar_wait(&s_done, 0);           // every key and every warp's min / max of the row has landed in this CTA
    SEL_CYC(5);
    uint32_t kmin = 0xFFFFFFFFu, kmax = 0u;
    for (int i = lane; i < (int)CS * NW; i += 32) { kmin = min(kmin, s_mm[i][0]); kmax = max(kmax, s_mm[i][1]); }
    kmin = __reduce_min_sync(0xffffffffu, kmin);
    kmax = __reduce_max_sync(0xffffffffu, kmax);

    // =============================== a2 (CTA 0, consumer threads): exact top-k, ascending ids ===============================
    topk_emit(s_keys, p.n_cand, p.topk, kmin, kmax, ids_row, p.slot_ids ? s_plan.nw : nullptr, s_hist, s_wtot, s_bcast, s_cand, cyc_);
    SEL_CYC(12);
    SEL_LOG_EXIT
    if (p.slot_ids) {
        consumer_sync();   // the row's k ids (n_cand > k: exactly k) are in s_plan.nw as well as on their way to global memory
        if (w == 0) {
            const int nm = reuse_plan_row(nullptr, p.slot_ids + (size_t)r * p.topk, plan_old, p.fetch + (size_t)r * p.topk, p.topk, s_plan, lane);
            if (lane == 0 && p.n_fetch) p.n_fetch[r] = nm;
            if (p.door) {
                __syncwarp();
                if (lane == 0) door_ring(p.door);
            }
        }
    } else if (p.door) {
        consumer_sync();   // every consumer thread has issued its ids
        if (tid == 0) door_ring(p.door);
    }
}

// a0: Kpool[r,j,d] = bf16( (1/S) sum_t K[r,j,t,d] ), fp32 sum in ascending t (Eq.2, kernel = stride = S).
// D/8 lanes per block, each lane owns 8 consecutive d and walks the 64 tokens in order.
template <int D>
__global__ void __launch_bounds__(256) pool_keys_kernel(const uint4* __restrict__ kv, uint4* __restrict__ kpool,
                                                         int64_t n_rb /* rows*blocks */) {
    constexpr int LPK = D / 8, S = 64;
    const int64_t gthread = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t rb = gthread / LPK;
    const int dl = (int)(gthread % LPK);
    if (rb >= n_rb) return;
    const uint4* src = kv + rb * (2 * S * LPK) + dl;  // plane 0 = K
    float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#pragma unroll 8
    for (int t = 0; t < S; ++t) {
        uint4 v = __ldg(src + (size_t)t * LPK);
        acc[0] += bf16_lo(v.x); acc[1] += bf16_hi(v.x); acc[2] += bf16_lo(v.y); acc[3] += bf16_hi(v.y);
        acc[4] += bf16_lo(v.z); acc[5] += bf16_hi(v.z); acc[6] += bf16_lo(v.w); acc[7] += bf16_hi(v.w);
    }
    const float inv = 1.0f / S;
    uint4 o;
    o.x = pack_bf16(acc[0] * inv, acc[1] * inv);
    o.y = pack_bf16(acc[2] * inv, acc[3] * inv);
    o.z = pack_bf16(acc[4] * inv, acc[5] * inv);
    o.w = pack_bf16(acc[6] * inv, acc[7] * inv);
    kpool[rb * LPK + dl] = o;
}

// a0 for f3: compressed keys with overlapping windows, Eq.2 with (l_C, s) = (32, 16):
// Kgrid[r,j,:] = bf16( (1/32) sum_{t=16j}^{16j+31} K[r,t,:] ), fp32 sum in ascending t; j < n_comp = T/16 - 1, the
// remaining row of the [R][4*Nb][D] grid is zero.  D/8 lanes per compressed key.
template <int D>
__global__ void __launch_bounds__(256) pool_keys_grid_kernel(const uint4* __restrict__ kv, uint4* __restrict__ kgrid, int n_blocks,
                                                              int64_t n_rj /* rows * 4 * n_blocks */) {
    constexpr int LPK = D / 8, S = 64, WIN = 32, STR = 16;
    const int64_t gthread = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t rj = gthread / LPK;
    const int dl = (int)(gthread % LPK);
    if (rj >= n_rj) return;
    const int per_row = n_blocks * (S / STR);
    const int64_t r = rj / per_row;
    const int j = (int)(rj % per_row);
    uint4 o = make_uint4(0, 0, 0, 0);
    if (j < per_row - 1) {
        float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#pragma unroll 8
        for (int i = 0; i < WIN; ++i) {
            const int t = j * STR + i;
            const uint4 v = __ldg(kv + ((r * n_blocks + t / S) * 2 * S + (t % S)) * LPK + dl);   // plane 0 = K
            acc[0] += bf16_lo(v.x); acc[1] += bf16_hi(v.x); acc[2] += bf16_lo(v.y); acc[3] += bf16_hi(v.y);
            acc[4] += bf16_lo(v.z); acc[5] += bf16_hi(v.z); acc[6] += bf16_lo(v.w); acc[7] += bf16_hi(v.w);
        }
        const float inv = 1.0f / WIN;
        o.x = pack_bf16(acc[0] * inv, acc[1] * inv);
        o.y = pack_bf16(acc[2] * inv, acc[3] * inv);
        o.z = pack_bf16(acc[4] * inv, acc[5] * inv);
        o.w = pack_bf16(acc[6] * inv, acc[7] * inv);
    }
    kgrid[rj * LPK + dl] = o;
}

// f2, Alg.2 lines 2-3: append the new token's K and V at position t of every row's cache (device-resident, or
// pinned host memory written through UVA: the asynchronous write-back of P:L159) and update the pooled keys incrementally
// (P:L89): ksum accumulates the open block's keys in fp32 in arrival (= ascending t) order, exactly the sum order of
// pool_keys_kernel, so the pooled key written when the block completes is bit-identical to pooling the finished block.
template <int D>
__global__ void __launch_bounds__(256) append_kv_kernel(const uint4* __restrict__ k_new, const uint4* __restrict__ v_new,
                                                         uint4* __restrict__ kv, float* __restrict__ ksum, uint4* __restrict__ kpool,
                                                         int n_rows, int n_blocks, int64_t t) {
    constexpr int LPK = D / 8, S = 64;
    const int gthread = blockIdx.x * blockDim.x + threadIdx.x;
    const int r = gthread / LPK, dl = gthread % LPK;
    if (r >= n_rows) return;
    const int64_t j = t / S;
    const int o = (int)(t % S);
    const uint4 k = __ldg(k_new + (size_t)r * LPK + dl), v = __ldg(v_new + (size_t)r * LPK + dl);
    uint4* blk = kv + ((size_t)r * n_blocks + j) * (2 * S * LPK);
    blk[(size_t)o * LPK + dl] = k;                      // plane 0 = K
    blk[(size_t)(S + o) * LPK + dl] = v;                // plane 1 = V
    float* acc = ksum + ((size_t)r * LPK + dl) * 8;
    float a[8];
    const float4 a0 = *reinterpret_cast<const float4*>(acc), a1 = *reinterpret_cast<const float4*>(acc + 4);
    a[0] = a0.x + bf16_lo(k.x); a[1] = a0.y + bf16_hi(k.x); a[2] = a0.z + bf16_lo(k.y); a[3] = a0.w + bf16_hi(k.y);
    a[4] = a1.x + bf16_lo(k.z); a[5] = a1.y + bf16_hi(k.z); a[6] = a1.z + bf16_lo(k.w); a[7] = a1.w + bf16_hi(k.w);
    if (o == S - 1) {
        const float inv = 1.0f / S;
        uint4 p;
        p.x = pack_bf16(a[0] * inv, a[1] * inv);
        p.y = pack_bf16(a[2] * inv, a[3] * inv);
        p.z = pack_bf16(a[4] * inv, a[5] * inv);
        p.w = pack_bf16(a[6] * inv, a[7] * inv);
        kpool[((size_t)r * n_blocks + j) * LPK + dl] = p;
#pragma unroll
        for (int i = 0; i < 8; ++i) a[i] = 0.f;
    }
    *reinterpret_cast<float4*>(acc) = make_float4(a[0], a[1], a[2], a[3]);
    *reinterpret_cast<float4*>(acc + 4) = make_float4(a[4], a[5], a[6], a[7]);
}

}  // namespace

// Cluster size of the select launch (measured on B200 at 128K, batch 4 .. 128, cold HBM): the largest power of two <= 8 such
// that every CTA has at least one stage of keys, R*CS <= SM count (one CTA per SM: 64 .. 128 CTAs stream as fast as 256, and
// twice the CTAs only add to the cluster barrier and to the launch) and the device can keep all R clusters resident at once
// (asked once per context, cluster size and shared-memory size).  16-CTA clusters lose to 8 at every batch (barrier cost,
// non-portable placement).  With more rows than SMs one CTA per row runs two to an SM and in waves, and the selection of one
// row overlaps the stream of the next.
template <int D, bool GRID>
static int select_launch(sparda_ctx* ctx, const void* Kpool, const SelParams& p0, cudaStream_t st) {
    auto kern = forecast_select_kernel<D, GRID>;
    constexpr int KPB = GRID ? 4 : 1;
    constexpr int CPS = SEL_STAGE_BYTES / (D * 2) / KPB;   // candidates per stage
    sparda_kernel_state& ks = ctx->kstate[(GRID ? SPARDA_K_SELECT_GRID_128 : SPARDA_K_SELECT_128) + (D == 128 ? 0 : 1)];
    if (!ks.attr_set) {
        SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 8192));
        SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        ks.attr_set = true;
    }
    SelParams p = p0;
    // key array in CTA 0: sized in steps of 2048 candidates so that the occupancy answers below stay valid
    const size_t key_bytes = p.n_cand > p.topk ? (size_t)((p.n_cand + 2047) & ~2047) * sizeof(uint32_t) : 0;
    const size_t smem = 1023 + (size_t)SEL_STAGES * SEL_STAGE_BYTES + key_bytes;
    if (smem > 227 * 1024 - 8192) return SPARDA_EINVAL;
    CUtensorMap map;
    int rc = sparda_get_tmap(ctx, Kpool, (uint64_t)ctx->R * p.n_blocks * KPB, D, 64, &map);
    if (rc) return rc;
    cudaLaunchConfig_t lc = {};
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    at[1] = sparda_pdl_attr();
    lc.attrs = at;
    lc.numAttrs = sparda_use_pdl(ctx) ? 2 : 1;
    lc.blockDim = dim3(SEL_CTA_THREADS, 1, 1);
    lc.dynamicSmemBytes = smem;
    lc.stream = st;
    int cs = 1;
    if (p.n_cand > p.topk) {
        const int n_stages = (p.n_cand + CPS - 1) / CPS;
        for (int c = ctx->cfg.select_cluster > 0 ? ctx->cfg.select_cluster : 8; c > 1; c /= 2) {
            if (ctx->cfg.select_cluster == 0 && (c > n_stages || (long long)ctx->R * c > ctx->sm_count)) continue;
            if (ks.max_clusters[c] == 0 || ks.asked_smem[c] != (int)smem) {
                int n = 0;
                lc.gridDim = dim3(c, 1, 1);
                at[0].val.clusterDim.x = c;
                const unsigned na = lc.numAttrs;
                lc.numAttrs = 1;
                cudaError_t e = cudaOccupancyMaxActiveClusters(&n, kern, &lc);
                lc.numAttrs = na;
                (void)cudaGetLastError();
                ks.max_clusters[c] = (e == cudaSuccess && n >= 1) ? n : -1;
                ks.asked_smem[c] = (int)smem;
            }
            if (ks.max_clusters[c] >= (ctx->cfg.select_cluster > 0 ? 1 : ctx->R)) { cs = c; break; }
        }
    }
    p.per = (p.n_cand + cs - 1) / cs;
    lc.gridDim = dim3((unsigned)(ctx->R * cs), 1, 1);
    at[0].val.clusterDim.x = cs;
    SPARDA_CUDA_TRY(ctx, cudaLaunchKernelEx(&lc, kern, map, p));
    ctx->last_select_cluster = cs;
    return SPARDA_OK;
}

int sparda_launch_select(sparda_ctx* ctx, const void* F, const void* Kpool, int n_blocks, int n_cand, int topk,
                         int32_t* ids, int32_t* slot_ids, int32_t* fetch, int32_t* n_fetch, cudaStream_t st) {
    if (slot_ids && topk > RP_MAXK) return SPARDA_EINVAL;
    SelParams p;
    p.slot_ids = slot_ids;
    p.fetch = fetch;
    p.n_fetch = n_fetch;
    p.door = ctx->door_next;
    p.F = (const uint32_t*)F;
    p.ids = ids;
    p.n_blocks = n_blocks;
    p.n_cand = n_cand;
    p.topk = topk;
    p.per = n_cand;
    p.keys_valid = n_cand;
    p.n_init = p.n_local = 0;
    int rc = ctx->cfg.head_dim == 128 ? select_launch<128, false>(ctx, Kpool, p, st) : select_launch<64, false>(ctx, Kpool, p, st);
    if (rc) return rc;
    ctx->launches++;
    return SPARDA_OK;
}

// f3: the same launch over the (32,16) compressed-key grid [R][4*n_blocks][D] with the max-pool to blocks and the
// init / local blocks forced in (reading q19).
int sparda_launch_select_grid(sparda_ctx* ctx, const void* F, const void* Kgrid, int n_blocks, int n_cand, int n_init, int n_local,
                              int topk, int32_t* ids, cudaStream_t st) {
    SelParams p;
    p.slot_ids = p.fetch = p.n_fetch = nullptr;
    p.door = ctx->door_next;
    p.F = (const uint32_t*)F;
    p.ids = ids;
    p.n_blocks = n_blocks;
    p.n_cand = n_cand;
    p.topk = topk;
    p.per = n_cand;
    p.keys_valid = 4 * n_cand - 1;
    p.n_init = n_init;
    p.n_local = n_local;
    int rc = ctx->cfg.head_dim == 128 ? select_launch<128, true>(ctx, Kgrid, p, st) : select_launch<64, true>(ctx, Kgrid, p, st);
    if (rc) return rc;
    ctx->launches++;
    return SPARDA_OK;
}

int sparda_launch_pool_keys(sparda_ctx* ctx, const void* kv, int64_t n_rows, int n_blocks, void* kpool, cudaStream_t st) {
    const int64_t n_rb = n_rows * n_blocks;
    const int lpk = ctx->cfg.head_dim / 8;
    const int64_t threads = n_rb * lpk;
    const unsigned grid = (unsigned)((threads + 255) / 256);
    if (ctx->cfg.head_dim == 128)
        pool_keys_kernel<128><<<grid, 256, 0, st>>>((const uint4*)kv, (uint4*)kpool, n_rb);
    else
        pool_keys_kernel<64><<<grid, 256, 0, st>>>((const uint4*)kv, (uint4*)kpool, n_rb);
    SPARDA_CUDA_TRY(ctx, cudaGetLastError());
    ctx->launches++;
    return SPARDA_OK;
}

int sparda_launch_append_kv(sparda_ctx* ctx, const void* k_new, const void* v_new, int64_t t, void* kv, int n_blocks, float* ksum,
                            void* kpool, cudaStream_t st) {
    const int lpk = ctx->cfg.head_dim / 8;
    const int threads = ctx->R * lpk;
    const unsigned grid = (unsigned)((threads + 255) / 256);
    if (ctx->cfg.head_dim == 128)
        append_kv_kernel<128><<<grid, 256, 0, st>>>((const uint4*)k_new, (const uint4*)v_new, (uint4*)kv, ksum, (uint4*)kpool, ctx->R, n_blocks, t);
    else
        append_kv_kernel<64><<<grid, 256, 0, st>>>((const uint4*)k_new, (const uint4*)v_new, (uint4*)kv, ksum, (uint4*)kpool, ctx->R, n_blocks, t);
    SPARDA_CUDA_TRY(ctx, cudaGetLastError());
    ctx->launches++;
    return SPARDA_OK;
}

int sparda_launch_pool_keys_grid(sparda_ctx* ctx, const void* kv, int64_t n_rows, int n_blocks, void* kgrid, cudaStream_t st) {
    const int64_t n_rj = n_rows * n_blocks * 4;
    const int lpk = ctx->cfg.head_dim / 8;
    const unsigned grid = (unsigned)((n_rj * lpk + 255) / 256);
    if (ctx->cfg.head_dim == 128)
        pool_keys_grid_kernel<128><<<grid, 256, 0, st>>>((const uint4*)kv, (uint4*)kgrid, n_blocks, n_rj);
    else
        pool_keys_grid_kernel<64><<<grid, 256, 0, st>>>((const uint4*)kv, (uint4*)kgrid, n_blocks, n_rj);
    SPARDA_CUDA_TRY(ctx, cudaGetLastError());
    ctx->launches++;
    return SPARDA_OK;
}
