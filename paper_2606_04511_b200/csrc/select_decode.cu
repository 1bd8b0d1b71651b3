// Forecast indexer for decode (a1 + a2) and key compression (a0).
//
//   s[r,j] = sum_d F[r,d] * Kpool[r,j,d]      Eq.4: raw logits, no softmax, no scale
//   ids[r] = f_top(s[r, 0:n_cand], k)          P:L78: k best blocks, ties -> lowest id, ascending ids, -1 padded
//
// One launch, one thread-block cluster per row r.  The row's n_cand pooled keys are cut into CS contiguous ranges,
// one per CTA of the cluster (CS = 1..16, chosen so that R*CS fills the SMs).  In every CTA a producer warp streams
// its range through a ring of 16 KiB shared-memory stages with bulk copies (TMA engine, cp.async.bulk on
// mbarriers: 96 KiB in flight per CTA, two CTAs per SM, no registers or LSU slots spent on the stream); 8 consumer warps take the
// dot products out of shared memory (D/8 lanes per key, 16-byte conflict-free reads, fp32 FMA, shuffle reduction)
// and store order-preserving uint32 keys straight into the shared memory of the cluster's CTA 0 (DSMEM), together
// with per-warp min / max.  After one cluster barrier CTA 0 holds the whole row's scores on chip and selects: a
// one-pass 256-bucket value histogram finds the boundary bucket of the k-th largest, one warp ranks its few members
// exactly, and an index-ordered compaction emits {key > T} plus the first (k - #{key > T}) keys == T, which is
// exactly "sort by (score desc, id asc), take k, sort by id".  Scores never touch global memory; there is no
// ticket, no fence and no scratch.  HBM-bound: R*n_cand*D*2 bytes of Kpool.
#include "sparda_internal.cuh"
#include "reuse_plan.cuh"
#ifdef SEL_CS_ENV
#include <cstdlib>
#endif

#ifdef SPARDA_TRACE
__device__ unsigned long long* g_sel_trace;   // [gridDim.x][16] globaltimer stamps (debug builds only)
extern "C" void sparda_debug_set_sel_trace(unsigned long long* p) { cudaMemcpyToSymbol(g_sel_trace, &p, sizeof(p)); }
#define SEL_TRACE(i)                                                                          \
    if (threadIdx.x == 0) {                                                                   \
        unsigned long long t__;                                                               \
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t__));                               \
        g_sel_trace[blockIdx.x * 16 + (i)] = t__;                                              \
    }
#else
#define SEL_TRACE(i)
#endif

namespace {

using namespace sparda;

constexpr int SEL_THREADS = 256;                  // consumer threads (the selection runs on these)
constexpr int SEL_CTA_THREADS = SEL_THREADS + 32; // + one producer warp
#ifndef SEL_STAGE_BYTES_V
#define SEL_STAGE_BYTES_V 16384
#define SEL_STAGES_V 6
#endif
constexpr int SEL_STAGE_BYTES = SEL_STAGE_BYTES_V;
constexpr int SEL_STAGES = SEL_STAGES_V;
constexpr int SEL_MAX_CS = 16;                    // largest cluster (non-portable size, opt-in)

// barrier of the 256 consumer threads only (the producer warp has left by the time the selection runs)
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive1(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
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
__device__ __forceinline__ void st_cluster_u32(uint32_t addr, uint32_t v) {
    asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
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
    return __uint_as_float(key ^ ((key >> 31) ? 0x80000000u : 0xFFFFFFFFu));
}

constexpr int SEL_CAND_CAP = 32;  // boundary-bucket size the one-warp exact finish handles

// Exact top-k over keys[0..n) (order-preserving uint32 keys in shared memory), k < n <= 8192.  256 consumer threads.
//
// Fast path, three CTA barriers:
//  1. one histogram pass over 256 equal-width value buckets of the row's [min, max] (hist is zeroed by the caller).
//     The bucket map is monotone (subtract, multiply by a positive constant, truncate: all monotone under IEEE
//     rounding), so every key in a higher bucket is larger than every key in a lower one and equal keys share a
//     bucket.  Unlike a radix pass over the top byte of the key (sign + 7 exponent bits: a handful of bins for
//     Gaussian logits) the shared-memory atomics are spread.
//  2. every warp redundantly suffix-scans the 256 counts (8 per lane + one shuffle scan) and finds the boundary bucket
//     b* holding the k-th largest -- no broadcast, no barrier.  Each thread then walks its contiguous slice of the row
//     once: keys above b* are selected (a bit mask in a register), members of b* (<= 32, typically ~4) go to a list.
//  3. every warp redundantly ranks the list by (key desc, id asc) with shuffles, which yields the k-th largest key and
//     the largest id taken among its equals; a thread completes its mask, one block scan of the counts places it, and
//     the ids are emitted in index order: exactly "sort by (score desc, id asc), take k, sort by id".
// Fallback (heavy ties / degenerate range): exact MSB-first 8-bit radix select + index-ordered compaction.
__device__ void topk_emit(const uint32_t* keys, int n, int k, uint32_t kmin, uint32_t kmax, int32_t* ids_out,
                          uint32_t* hist /*[256], zeroed*/, uint32_t* warp_tot /*[8]*/, uint32_t* bcast /*[4], [2] zeroed*/,
                          uint32_t* cand /*[2 * SEL_CAND_CAP]*/) {
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int per = (n + SEL_THREADS - 1) / SEL_THREADS;          // <= 32: a thread's slice fits one bit mask
    const int lo = min(tid * per, n), hi = min(lo + per, n);
    const float flo = key_to_float(kmin), fhi = key_to_float(kmax);
    const float scale = 256.0f / (fhi - flo);
    bool fast = (kmax > kmin) && (scale > 0.f) && (scale < INFINITY);
    auto bucket = [&](uint32_t key) -> int {
        return (int)fminf((key_to_float(key) - flo) * scale, 255.0f);
    };
    if (fast) {
        SEL_TRACE(4);
        for (int i = tid; i < n; i += SEL_THREADS) atomicAdd(&hist[bucket(keys[i])], 1u);
        consumer_sync();
        SEL_TRACE(5);
        // suffix counts, redundantly per warp: lane l owns buckets 255 - 8l - j, j = 0..7 (descending value)
        uint32_t h[8], run = 0;
#pragma unroll
        for (int j = 0; j < 8; ++j) { h[j] = hist[255 - 8 * lane - j]; run += h[j]; }
        uint32_t incl = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t nb = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += nb;
        }
        uint32_t gt = incl - run;                                 // keys in buckets above this lane's eight
        int my_b = -1;
        uint32_t my_need = 0, my_pop = 0;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            if (gt < (uint32_t)k && (uint32_t)k <= gt + h[j]) { my_b = 255 - 8 * lane - j; my_need = k - gt; my_pop = h[j]; }
            gt += h[j];
        }
        const int src = __ffs(__ballot_sync(0xffffffffu, my_b >= 0)) - 1;   // exactly one lane (n > k)
        const int bstar = __shfl_sync(0xffffffffu, my_b, src);
        const uint32_t need = __shfl_sync(0xffffffffu, my_need, src), pop = __shfl_sync(0xffffffffu, my_pop, src);
        SEL_TRACE(6);
        if (pop <= SEL_CAND_CAP) {
            uint32_t m_sel = 0, m_eq = 0;
            for (int i = lo; i < hi; ++i) {
                const uint32_t key = keys[i];
                const int b = bucket(key);
                if (b > bstar) m_sel |= 1u << (i - lo);
                if (b == bstar) {
                    m_eq |= 1u << (i - lo);
                    const uint32_t s = atomicAdd(&bcast[2], 1u);
                    cand[2 * s] = key;
                    cand[2 * s + 1] = (uint32_t)i;
                }
            }
            consumer_sync();
            SEL_TRACE(7);
            // rank the boundary bucket, redundantly per warp: lane i holds member i
            const bool have = (uint32_t)lane < pop;
            const uint32_t mk = have ? cand[2 * lane] : 0u, mi = have ? cand[2 * lane + 1] : 0xFFFFFFFFu;
            uint32_t rank = 0;
            for (uint32_t f = 0; f < pop; ++f) {
                const uint32_t fk = __shfl_sync(0xffffffffu, mk, f), fi = __shfl_sync(0xffffffffu, mi, f);
                rank += (fk > mk || (fk == mk && fi < mi)) ? 1u : 0u;
            }
            const int ks = __ffs(__ballot_sync(0xffffffffu, have && rank == need - 1)) - 1;   // the k-th largest of the row
            const uint32_t Tk = __shfl_sync(0xffffffffu, mk, ks), Ti = __shfl_sync(0xffffffffu, mi, ks);
            SEL_TRACE(8);
            while (m_eq) {
                const int j = __ffs(m_eq) - 1;
                m_eq &= m_eq - 1;
                const uint32_t key = keys[lo + j];
                if (key > Tk || (key == Tk && (uint32_t)(lo + j) <= Ti)) m_sel |= 1u << j;
            }
            // place and emit
            const uint32_t c = __popc(m_sel);
            uint32_t inc = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t nb = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += nb;
            }
            if (lane == 31) warp_tot[w] = inc;
            consumer_sync();
            SEL_TRACE(9);
            uint32_t pos = inc - c;
#pragma unroll
            for (int i = 0; i < SEL_THREADS / 32; ++i) pos += i < w ? warp_tot[i] : 0u;
            while (m_sel) {
                const int j = __ffs(m_sel) - 1;
                m_sel &= m_sel - 1;
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
            ids_out[pos++] = i;
        } else if (key == T) {
            if (eq_before < krem) ids_out[pos++] = i;
            ++eq_before;
        }
    }
}


struct SelParams {
    const uint4* F;
    const char* Kpool;
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
};

template <int D, bool GRID>
__global__ void __launch_bounds__(SEL_CTA_THREADS, 1) forecast_select_kernel(SelParams p) {
    constexpr int KPB = GRID ? 4 : 1;                // keys per candidate block
    constexpr int LPK = D / 8;                       // lanes per key (16 B = 8 bf16 each)
    constexpr int KPL = 32 / LPK;                    // keys per warp-wide read
    constexpr int NW = SEL_THREADS / 32;
    constexpr int ROW_BYTES = D * 2;
    constexpr int KPS = SEL_STAGE_BYTES / ROW_BYTES; // keys per stage
    constexpr int PASSES = KPS / (NW * KPL);
    extern __shared__ uint8_t sel_smem_raw[];
    __shared__ uint64_t s_full[SEL_STAGES], s_empty[SEL_STAGES];
    __shared__ uint32_t s_hist[256];
    __shared__ uint32_t s_wtot[8];
    __shared__ uint32_t s_bcast[4];
    __shared__ uint32_t s_cand[2 * SEL_CAND_CAP];
    __shared__ uint32_t s_mm[2][SEL_MAX_CS * NW];    // per (CTA of the cluster, warp): min / max key; lives in CTA 0
    __shared__ ReusePlanScratch s_plan;

    uint8_t* ring = (uint8_t*)(((uintptr_t)sel_smem_raw + 127) & ~(uintptr_t)127);
    uint32_t* s_keys = reinterpret_cast<uint32_t*>(ring + SEL_STAGES * SEL_STAGE_BYTES);   // [n_cand], used in CTA 0

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const uint32_t c = cluster_ctarank();
    uint32_t CS;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(CS));
    const int r = blockIdx.x / CS;
    int32_t* ids_row = p.ids + (size_t)r * p.topk;

    if (p.n_cand <= p.topk) {  // every candidate is selected (reading q5); no scoring needed
        if (c == 0) {
            for (int i = tid; i < p.topk; i += SEL_CTA_THREADS) ids_row[i] = i < p.n_cand ? i : -1;
            if (p.slot_ids) {
                __syncthreads();
                if (w == 0) {
                    const int nm = reuse_plan_row(ids_row, p.slot_ids + (size_t)r * p.topk, p.fetch + (size_t)r * p.topk, p.topk, s_plan, lane);
                    if (lane == 0 && p.n_fetch) p.n_fetch[r] = nm;
                }
            }
        }
        return;
    }

    if (tid == 0) {
        for (int s = 0; s < SEL_STAGES; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], NW); }
        mbar_fence_init();
        fence_proxy_async_smem();
    }
    __syncthreads();
    SEL_TRACE(0);

    const int k_lo = min((int)c * p.per, p.n_cand);
    const int n_local = min(p.per, p.n_cand - k_lo);
    const int n_keys_local = n_local * KPB;         // rows of Kpool this CTA streams
    const int n_st = (n_keys_local + KPS - 1) / KPS;

    if (w == NW) {
        // =============================== producer warp: bulk copies into the ring ===============================
        if (lane == 0) {
            const char* src = p.Kpool + ((size_t)r * p.n_blocks + k_lo) * KPB * ROW_BYTES;
            for (int i = 0; i < n_st; ++i) {
                const int s = i % SEL_STAGES;
                if (i >= SEL_STAGES) mbar_wait(&s_empty[s], ((i / SEL_STAGES) - 1) & 1);
                const uint32_t bytes = (uint32_t)min(KPS, n_keys_local - i * KPS) * ROW_BYTES;
                mbar_arrive_expect_tx(&s_full[s], bytes);
                bulk_g2s(ring + (size_t)s * SEL_STAGE_BYTES, src + (size_t)i * SEL_STAGE_BYTES, bytes, &s_full[s]);
            }
        }
    } else {
        // =============================== consumers: a1, scores of this CTA's range ===============================
        const int sub = lane / LPK, dl = lane % LPK;
        const uint4 fv = __ldg(p.F + (size_t)r * LPK + dl);
        float f[8];
        f[0] = bf16_lo(fv.x); f[1] = bf16_hi(fv.x); f[2] = bf16_lo(fv.y); f[3] = bf16_hi(fv.y);
        f[4] = bf16_lo(fv.z); f[5] = bf16_hi(fv.z); f[6] = bf16_lo(fv.w); f[7] = bf16_hi(fv.w);
        const uint32_t keys0 = map_to_cta(s_keys, 0);          // the row's key array lives in CTA 0
        uint32_t kmin = 0xFFFFFFFFu, kmax = 0u;
        for (int i = 0; i < n_st; ++i) {
            const int s = i % SEL_STAGES;
            const int nk = min(KPS, n_keys_local - i * KPS);
            mbar_wait(&s_full[s], (i / SEL_STAGES) & 1);
            const uint8_t* st = ring + (size_t)s * SEL_STAGE_BYTES;
            uint4 kv[PASSES];
#pragma unroll
            for (int ps = 0; ps < PASSES; ++ps) {
                // plain: pass ps takes key ps*16 + group; grid: the group takes the 4 keys of one block, one per pass
                const int kl = GRID ? (w * KPL + sub) * 4 + ps : ps * (NW * KPL) + w * KPL + sub;
                kv[ps] = kl < nk ? *reinterpret_cast<const uint4*>(st + (size_t)kl * ROW_BYTES + dl * 16) : make_uint4(0, 0, 0, 0);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive1(&s_empty[s]);            // the stage is in registers: hand it back
#ifdef SEL_NOCOMPUTE
            if (kv[0].x == 0x12345678u) kmin = 0;
            continue;
#endif
            float sc[PASSES];
#pragma unroll
            for (int ps = 0; ps < PASSES; ++ps) {
                float a = f[0] * bf16_lo(kv[ps].x);
                a = fmaf(f[1], bf16_hi(kv[ps].x), a);
                a = fmaf(f[2], bf16_lo(kv[ps].y), a);
                a = fmaf(f[3], bf16_hi(kv[ps].y), a);
                a = fmaf(f[4], bf16_lo(kv[ps].z), a);
                a = fmaf(f[5], bf16_hi(kv[ps].z), a);
                a = fmaf(f[6], bf16_lo(kv[ps].w), a);
                sc[ps] = fmaf(f[7], bf16_hi(kv[ps].w), a);
            }
            // Transposed butterfly over the LPK lanes of a key: instead of reducing each of the 4 partial sums over all
            // lanes (4 * log2(LPK) shuffles), the two highest lane bits split the 4 sums between the lanes (2 + 1
            // shuffles), the remaining bits are plain butterflies on the one sum a lane is left with.  Pass `mine` of
            // the stage ends up complete in the lanes whose two highest key-lane bits spell `mine`.
            static_assert(PASSES == 4 && LPK >= 4, "the transposed reduction is written for 4 partial sums per lane");
            const bool hi1 = (dl & (LPK / 2)) != 0, hi2 = (dl & (LPK / 4)) != 0;
            const float r0 = __shfl_xor_sync(0xffffffffu, hi1 ? sc[0] : sc[2], LPK / 2);
            const float r1 = __shfl_xor_sync(0xffffffffu, hi1 ? sc[1] : sc[3], LPK / 2);
            const float v0 = (hi1 ? sc[2] : sc[0]) + r0, v1 = (hi1 ? sc[3] : sc[1]) + r1;
            float tot = (hi2 ? v1 : v0) + __shfl_xor_sync(0xffffffffu, hi2 ? v0 : v1, LPK / 4);
#pragma unroll
            for (int o = LPK / 8; o >= 1; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
            const int mine = (hi1 ? 2 : 0) + (hi2 ? 1 : 0);
            if (GRID) {
                // f_top's max-pool (reading q19): block score = max over the compressed keys that start in the block
                const int blk = i * (KPS / 4) + w * KPL + sub;                     // block within this CTA's range
                const int jkey = (k_lo + blk) * 4 + mine;                            // compressed key index in the row
                float bsc = jkey < p.keys_valid ? tot : -INFINITY;
                bsc = fmaxf(bsc, __shfl_xor_sync(0xffffffffu, bsc, LPK / 2));
                bsc = fmaxf(bsc, __shfl_xor_sync(0xffffffffu, bsc, LPK / 4));
                if (dl == 0 && blk < n_local) {
                    const int b = k_lo + blk;
                    const bool forced = b < p.n_init || b >= p.n_cand - p.n_local;   // init / local blocks: always attended
                    const uint32_t key = forced ? 0xFFFFFFFFu : orderable(bsc + 0.0f);
                    st_cluster_u32(keys0 + 4u * (uint32_t)b, key);
                    if (!forced) { kmin = min(kmin, key); kmax = max(kmax, key); }
                }
            } else {
                const int kl = mine * (NW * KPL) + w * KPL + sub;
                if ((dl & (LPK / 4 - 1)) == 0 && kl < nk) {
                    const uint32_t key = orderable(tot + 0.0f);      // +0: -0 -> +0
                    st_cluster_u32(keys0 + 4u * (uint32_t)(k_lo + i * KPS + kl), key);
                    kmin = min(kmin, key);
                    kmax = max(kmax, key);
                }
            }
        }
        kmin = __reduce_min_sync(0xffffffffu, kmin);
        kmax = __reduce_max_sync(0xffffffffu, kmax);
        if (lane == 0) {
            st_cluster_u32(map_to_cta(&s_mm[0][c * NW + w], 0), kmin);
            st_cluster_u32(map_to_cta(&s_mm[1][c * NW + w], 0), kmax);
        }
    }
    if (tid < 256) s_hist[tid] = 0;
    if (tid == 0) s_bcast[2] = 0;
    SEL_TRACE(1);
    // every CTA's keys and min / max have landed in CTA 0 once the cluster barrier completes (release / acquire)
    cluster_sync_all();
    SEL_TRACE(2);
    if (c != 0 || w == NW) return;

    // =============================== a2 (CTA 0, consumer threads): exact top-k, ascending ids ===============================
    uint32_t kmin = 0xFFFFFFFFu, kmax = 0u;
    for (int i = lane; i < (int)CS * NW; i += 32) { kmin = min(kmin, s_mm[0][i]); kmax = max(kmax, s_mm[1][i]); }
    kmin = __reduce_min_sync(0xffffffffu, kmin);
    kmax = __reduce_max_sync(0xffffffffu, kmax);
    topk_emit(s_keys, p.n_cand, p.topk, kmin, kmax, ids_row, s_hist, s_wtot, s_bcast, s_cand);
    SEL_TRACE(3);
    if (p.slot_ids) {
        consumer_sync();   // the row's ids are in global memory (read back through L2)
        if (w == 0) {
            const int nm = reuse_plan_row(ids_row, p.slot_ids + (size_t)r * p.topk, p.fetch + (size_t)r * p.topk, p.topk, s_plan, lane);
            if (lane == 0 && p.n_fetch) p.n_fetch[r] = nm;
        }
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

// Cluster size of the select launch: the largest power of two <= 16 such that R*CS CTAs fit the SMs (the
// ring takes 96 KiB of shared memory), every CTA has at least one stage of keys, and the driver can co-schedule
// such a cluster (asked once per size; sizes above 8 are non-portable and need the opt-in attribute).  Measured on
// B200 (batch 32, 2048 blocks, cold HBM): a 6 x 16 KiB ring streams as fast as 10 stages and lets two CTAs share an
// SM, so with R > SM count the selection of one row overlaps the stream of the next.
template <int D, bool GRID>
static int select_launch(sparda_ctx* ctx, const SelParams& p0, cudaStream_t st) {
    auto kern = forecast_select_kernel<D, GRID>;
    constexpr int KPS = SEL_STAGE_BYTES / (D * 2) / (GRID ? 4 : 1);   // candidates per stage
    static bool attr_set = false;
    static int cluster_ok[SEL_MAX_CS + 1];   // 0 = not asked, 1 = schedulable, -1 = not
    const size_t smem_max = 127 + (size_t)SEL_STAGES * SEL_STAGE_BYTES + (size_t)ctx->cfg.max_blocks * sizeof(uint32_t);
    if (!attr_set) {
        SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 8192));
        SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        attr_set = true;
    }
    if (smem_max > 227 * 1024 - 8192) return SPARDA_EINVAL;
    SelParams p = p0;
    const size_t smem = 127 + (size_t)SEL_STAGES * SEL_STAGE_BYTES + (size_t)(p.n_cand > p.topk ? p.n_cand : 0) * sizeof(uint32_t);
    cudaLaunchConfig_t lc = {};
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    lc.attrs = at;
    lc.numAttrs = 1;
    lc.blockDim = dim3(SEL_CTA_THREADS, 1, 1);
    lc.dynamicSmemBytes = smem;
    lc.stream = st;
    int cs = 1;
    if (p.n_cand > p.topk)
        while (cs * 2 <= SEL_MAX_CS && (long long)ctx->R * cs * 2 <= ctx->sm_count && cs * 2 <= (p.n_cand + KPS - 1) / KPS) cs *= 2;
#ifdef SEL_CS_ENV
    if (getenv("SPARDA_SELECT_CS") && p.n_cand > p.topk) cs = atoi(getenv("SPARDA_SELECT_CS"));
#endif
    for (; cs > 1; cs /= 2) {
        if (cluster_ok[cs] == 0) {
            int n = 0;
            lc.gridDim = dim3(cs, 1, 1);
            at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
            lc.dynamicSmemBytes = smem_max;
            cudaError_t e = cudaOccupancyMaxActiveClusters(&n, kern, &lc);
            (void)cudaGetLastError();
            cluster_ok[cs] = (e == cudaSuccess && n >= 1) ? 1 : -1;
            lc.dynamicSmemBytes = smem;
        }
        if (cluster_ok[cs] == 1) break;
    }
    p.per = (p.n_cand + cs - 1) / cs;
    lc.gridDim = dim3((unsigned)(ctx->R * cs), 1, 1);
    at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    SPARDA_CUDA_TRY(ctx, cudaLaunchKernelEx(&lc, kern, p));
    return SPARDA_OK;
}

int sparda_launch_select(sparda_ctx* ctx, const void* F, const void* Kpool, int n_blocks, int n_cand, int topk,
                         int32_t* ids, int32_t* slot_ids, int32_t* fetch, int32_t* n_fetch, cudaStream_t st) {
    if (slot_ids && topk > RP_MAXK) return SPARDA_EINVAL;
    SelParams p;
    p.slot_ids = slot_ids;
    p.fetch = fetch;
    p.n_fetch = n_fetch;
    p.F = (const uint4*)F;
    p.Kpool = (const char*)Kpool;
    p.ids = ids;
    p.n_blocks = n_blocks;
    p.n_cand = n_cand;
    p.topk = topk;
    p.per = n_cand;
    p.keys_valid = n_cand;
    p.n_init = p.n_local = 0;
    int rc = ctx->cfg.head_dim == 128 ? select_launch<128, false>(ctx, p, st) : select_launch<64, false>(ctx, p, st);
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
    p.F = (const uint4*)F;
    p.Kpool = (const char*)Kgrid;
    p.ids = ids;
    p.n_blocks = n_blocks;
    p.n_cand = n_cand;
    p.topk = topk;
    p.per = n_cand;
    p.keys_valid = 4 * n_cand - 1;
    p.n_init = n_init;
    p.n_local = n_local;
    int rc = ctx->cfg.head_dim == 128 ? select_launch<128, true>(ctx, p, st) : select_launch<64, true>(ctx, p, st);
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
