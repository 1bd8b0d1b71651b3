// Forecast indexer for decode (a1 + a2) and key compression (a0).
//
//   s[r,j] = sum_d F[r,d] * Kpool[r,j,d]      Eq.4: raw logits, no softmax, no scale
//   ids[r] = f_top(s[r, 0:n_cand], k)          P:L78: k best blocks, ties -> lowest id, ascending ids, -1 padded
//
// One launch.  Grid (chunks, R): each CTA streams a contiguous chunk of pooled keys with 16-byte
// coalesced loads (D/8 lanes per key, fp32 accumulate, shuffle reduction), writes order-preserving
// uint32 keys to an L2-resident scratch row, and takes a ticket; the last CTA of a row selects: an
// exact MSB-first 8-bit radix select finds the k-th largest key T, then an index-ordered compaction
// emits {key > T} plus the first (k - #{key > T}) entries with key == T, which is exactly
// "sort by (score desc, id asc), take k, sort by id".  HBM-bound: R*n_cand*D*2 bytes of Kpool.
#include "sparda_internal.cuh"

namespace {

using namespace sparda;

constexpr int SEL_THREADS = 256;
constexpr int SEL_KEYS_PER_CTA = 128;

__device__ __forceinline__ uint32_t block_incl_scan_256(uint32_t v, uint32_t* warp_tot /*[8]*/, uint32_t& total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t n = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += n;
    }
    if (lane == 31) warp_tot[w] = v;
    __syncthreads();
    uint32_t add = 0, tot = 0;
#pragma unroll
    for (int i = 0; i < SEL_THREADS / 32; ++i) {
        uint32_t t = warp_tot[i];
        if (i < w) add += t;
        tot += t;
    }
    total = tot;
    __syncthreads();
    return v + add;
}

__device__ __forceinline__ float key_to_float(uint32_t key) {
    return __uint_as_float(key ^ ((key >> 31) ? 0x80000000u : 0xFFFFFFFFu));
}

constexpr int SEL_CAND_CAP = 32;  // boundary-bucket size the one-warp exact finish handles

// Exact top-k over keys[0..n) (order-preserving uint32 keys in shared memory), n > k.  Whole CTA (256 threads).
//
// Fast path (one histogram pass): 256 equal-width value buckets over the row's [min, max]; the bucket map
// is monotone (subtract, multiply by a positive constant and truncate are all monotone under IEEE
// rounding), so every key in a higher bucket is larger than every key in a lower one and equal keys share
// a bucket.  A suffix scan finds the boundary bucket b* holding the k-th largest; its (<= 32, typically
// ~4) members are ranked exactly by (key desc, id asc) in one warp, which yields the k-th largest key T
// and how many keys == T are taken (the lowest ids).  Unlike a radix pass over the top byte of the key
// (sign + 7 exponent bits: a handful of bins for Gaussian logits) the shared-memory atomics are spread.
// Fallback (heavy ties / degenerate range): exact MSB-first 8-bit radix select.
// Emission: index-ordered compaction of {key > T} plus the first krem keys == T, which is exactly
// "sort by (score desc, id asc), take k, sort by id".
__device__ void topk_emit(const uint32_t* keys, int n, int k, uint32_t kmin, uint32_t kmax, int32_t* ids_out,
                          uint32_t* hist /*[256]*/, uint32_t* warp_tot /*[8]*/, uint32_t* bcast /*[4]*/,
                          uint32_t* cand /*[2 * SEL_CAND_CAP]*/) {
    const int tid = threadIdx.x;
    uint32_t T = 0, krem = 0;
    // ---- fast path
    const float flo = key_to_float(kmin), fhi = key_to_float(kmax);
    const float scale = 256.0f / (fhi - flo);
    bool fast = (kmax > kmin) && (scale > 0.f) && (scale < INFINITY);
    auto bucket = [&](uint32_t key) -> int {
        return (int)fminf((key_to_float(key) - flo) * scale, 255.0f);
    };
    if (fast) {
        hist[tid] = 0;
        if (tid == 0) bcast[2] = 0;
        __syncthreads();
        for (int i = tid; i < n; i += SEL_THREADS) atomicAdd(&hist[bucket(keys[i])], 1u);
        __syncthreads();
        // suffix sums: thread t owns bucket b = 255 - t; inclusive scan gives #keys with bucket >= b
        uint32_t mine = hist[255 - tid], tot;
        uint32_t ge = block_incl_scan_256(mine, warp_tot, tot);
        uint32_t gt = ge - mine;
        if (gt < (uint32_t)k && (uint32_t)k <= ge) {
            bcast[0] = 255 - tid;       // boundary bucket
            bcast[1] = k - gt;          // how many of its members are selected (>= 1)
            bcast[3] = mine;            // its population
        }
        __syncthreads();
        const int bstar = (int)bcast[0];
        const uint32_t need = bcast[1], pop = bcast[3];
        if (pop <= SEL_CAND_CAP) {
            for (int i = tid; i < n; i += SEL_THREADS) {
                uint32_t key = keys[i];
                if (bucket(key) == bstar) {
                    uint32_t s = atomicAdd(&bcast[2], 1u);
                    cand[2 * s] = key;
                    cand[2 * s + 1] = (uint32_t)i;
                }
            }
            __syncthreads();
            if (tid < 32) {
                const bool have = (uint32_t)tid < pop;
                const uint32_t mk = have ? cand[2 * tid] : 0u, mi = have ? cand[2 * tid + 1] : 0xFFFFFFFFu;
                uint32_t rank = 0;
                for (uint32_t f = 0; f < pop; ++f) {
                    const uint32_t fk = cand[2 * f], fi = cand[2 * f + 1];
                    rank += (fk > mk || (fk == mk && fi < mi)) ? 1u : 0u;
                }
                const bool is_kth = have && rank == need - 1;
                const uint32_t who = __ballot_sync(0xffffffffu, is_kth);   // exactly one lane
                const int src = __ffs(who) - 1;
                const uint32_t Tk = __shfl_sync(0xffffffffu, mk, src), Ti = __shfl_sync(0xffffffffu, mi, src);
                const uint32_t eq_taken = __popc(__ballot_sync(0xffffffffu, have && mk == Tk && mi <= Ti));
                if (tid == 0) { bcast[0] = Tk; bcast[1] = eq_taken; }
            }
            __syncthreads();
            T = bcast[0];
            krem = bcast[1];
        } else {
            fast = false;   // uniform across the CTA (pop is broadcast)
        }
        __syncthreads();
    }
    if (!fast) {
        uint32_t prefix = 0, mask = 0;
        krem = (uint32_t)k;
#pragma unroll 1
        for (int shift = 24; shift >= 0; shift -= 8) {
            hist[tid] = 0;
            __syncthreads();
            for (int i = tid; i < n; i += SEL_THREADS) {
                uint32_t key = keys[i];
                if ((key & mask) == prefix) atomicAdd(&hist[(key >> shift) & 255u], 1u);
            }
            __syncthreads();
            uint32_t mine = hist[255 - tid], tot;
            uint32_t ge = block_incl_scan_256(mine, warp_tot, tot);
            uint32_t gt = ge - mine;
            if (gt < krem && krem <= ge) {
                bcast[0] = prefix | ((uint32_t)(255 - tid) << shift);
                bcast[1] = krem - gt;
            }
            __syncthreads();
            prefix = bcast[0];
            krem = bcast[1];
            mask |= 0xFFu << shift;
            __syncthreads();
        }
        T = prefix;  // k-th largest key; take every key > T and the first `krem` keys == T
    }
    const int per = (n + SEL_THREADS - 1) / SEL_THREADS;
    const int lo = min(tid * per, n), hi = min(lo + per, n);
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

template <int D>
__global__ void __launch_bounds__(SEL_THREADS) forecast_select_kernel(const uint4* __restrict__ F,
                                                                       const uint4* __restrict__ Kpool,
                                                                       uint32_t* __restrict__ score_keys, int key_stride,
                                                                       unsigned int* __restrict__ tickets, int n_blocks,
                                                                       int n_cand, int topk, int32_t* __restrict__ ids) {
    constexpr int LPK = D / 8;         // lanes per key (16 B = 8 bf16 each)
    constexpr int KPL = 32 / LPK;      // keys per warp-wide load
    constexpr int NW = SEL_THREADS / 32;
    constexpr int ITERS = SEL_KEYS_PER_CTA / (NW * KPL);
    extern __shared__ uint32_t s_keys[];  // [n_cand] (only the selecting CTA uses it)
    __shared__ uint32_t s_hist[256];
    __shared__ uint32_t s_wtot[8];
    __shared__ uint32_t s_bcast[4];
    __shared__ uint32_t s_cand[2 * SEL_CAND_CAP];
    __shared__ uint32_t s_mm[2][SEL_THREADS / 32];
    __shared__ unsigned int s_ticket;

    const int r = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    int32_t* ids_row = ids + (size_t)r * topk;

    if (n_cand <= topk) {  // every candidate is selected (reading q5); no scoring needed
        if (blockIdx.x == 0)
            for (int i = tid; i < topk; i += SEL_THREADS) ids_row[i] = i < n_cand ? i : -1;
        return;
    }

    // ---- a1: scores of this CTA's chunk
    const int sub = lane / LPK, dl = lane % LPK;
    const uint4 fv = F[(size_t)r * LPK + dl];
    float f[8];
    f[0] = bf16_lo(fv.x); f[1] = bf16_hi(fv.x); f[2] = bf16_lo(fv.y); f[3] = bf16_hi(fv.y);
    f[4] = bf16_lo(fv.z); f[5] = bf16_hi(fv.z); f[6] = bf16_lo(fv.w); f[7] = bf16_hi(fv.w);
    const int j0 = blockIdx.x * SEL_KEYS_PER_CTA + w * (ITERS * KPL) + sub;
    const uint4* krow = Kpool + ((size_t)r * n_blocks) * LPK + dl;
    uint4 kv[ITERS];
#pragma unroll
    for (int it = 0; it < ITERS; ++it) {
        int j = j0 + it * KPL;
        kv[it] = j < n_cand ? __ldg(krow + (size_t)j * LPK) : make_uint4(0, 0, 0, 0);
    }
#pragma unroll
    for (int it = 0; it < ITERS; ++it) {
        float s = f[0] * bf16_lo(kv[it].x);
        s = fmaf(f[1], bf16_hi(kv[it].x), s);
        s = fmaf(f[2], bf16_lo(kv[it].y), s);
        s = fmaf(f[3], bf16_hi(kv[it].y), s);
        s = fmaf(f[4], bf16_lo(kv[it].z), s);
        s = fmaf(f[5], bf16_hi(kv[it].z), s);
        s = fmaf(f[6], bf16_lo(kv[it].w), s);
        s = fmaf(f[7], bf16_hi(kv[it].w), s);
#pragma unroll
        for (int o = LPK / 2; o >= 1; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        int j = j0 + it * KPL;
        if (dl == 0 && j < n_cand) score_keys[(size_t)r * key_stride + j] = orderable(s + 0.0f);  // +0: -0 -> +0
    }

    // ---- ticket: the last CTA of the row selects
    __threadfence();
    __syncthreads();
    if (tid == 0) s_ticket = atomicAdd(&tickets[r], 1u);
    __syncthreads();
    if (s_ticket != gridDim.x - 1) return;
    __threadfence();
    if (tid == 0) tickets[r] = 0;  // re-arm for the next launch
    uint32_t kmin = 0xFFFFFFFFu, kmax = 0u;
    for (int i = tid; i < n_cand; i += SEL_THREADS) {
        const uint32_t key = __ldcg(score_keys + (size_t)r * key_stride + i);
        s_keys[i] = key;
        kmin = min(kmin, key);
        kmax = max(kmax, key);
    }
    kmin = __reduce_min_sync(0xffffffffu, kmin);
    kmax = __reduce_max_sync(0xffffffffu, kmax);
    if (lane == 0) { s_mm[0][w] = kmin; s_mm[1][w] = kmax; }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < SEL_THREADS / 32; ++i) { kmin = min(kmin, s_mm[0][i]); kmax = max(kmax, s_mm[1][i]); }
    // ---- a2: exact top-k, ascending ids
    topk_emit(s_keys, n_cand, topk, kmin, kmax, ids_row, s_hist, s_wtot, s_bcast, s_cand);
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

}  // namespace

int sparda_launch_select(sparda_ctx* ctx, const void* F, const void* Kpool, int n_blocks, int n_cand, int topk,
                         int32_t* ids, cudaStream_t st) {
    const int chunks = n_cand > topk ? (n_cand + SEL_KEYS_PER_CTA - 1) / SEL_KEYS_PER_CTA : 1;
    dim3 grid(chunks, ctx->R);
    size_t smem = (size_t)(n_cand > topk ? n_cand : 0) * sizeof(uint32_t);
    if (ctx->cfg.head_dim == 128)
        forecast_select_kernel<128><<<grid, SEL_THREADS, smem, st>>>((const uint4*)F, (const uint4*)Kpool, (uint32_t*)ctx->scores,
                                                                      ctx->cfg.max_blocks, ctx->tickets, n_blocks, n_cand, topk, ids);
    else
        forecast_select_kernel<64><<<grid, SEL_THREADS, smem, st>>>((const uint4*)F, (const uint4*)Kpool, (uint32_t*)ctx->scores,
                                                                     ctx->cfg.max_blocks, ctx->tickets, n_blocks, n_cand, topk, ids);
    SPARDA_CUDA_TRY(ctx, cudaGetLastError());
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
