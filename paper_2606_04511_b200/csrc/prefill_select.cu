// Chunked-prefill selection (a7) and the multi-head softmax selector it replaces (a7').
//
//   a7  (Alg.1 l.2; Eq.4):  s[i,j] = F[g,i,:] . Kpool[g,j,:]  for the causal candidates
//        j < n_cand(i) = min(Nb, (i+1)/S)  (a block is visible once its last token <= i, reading q8),
//        ids[g,i] = f_top(s[i, 0:n_cand(i)], k): ties -> lowest id, ascending ids, -1 padded.
//   a7' (Eq.6 left):  s[i,j] = sum_{h in group g} softmax_j(Q[h,i,:] . Kpool[g,j,:] / sqrt(D)),
//        same causal candidates, same f_top.
//
// The Forecast-by-pooled-key product is a dense contraction ([T x D] x [D x Nb]), so it runs on the 5th-gen tensor
// cores: one persistent CTA per SM keeps its group's whole Kpool (Nb <= 512 rows, 128 KB at D = 128) resident in
// shared memory as the B operand, TMA-loads 128-row tiles of F (or Q_h) as the A operand (128-byte swizzle), and one
// elected thread issues tcgen05.mma (M = 128, N <= 256 per instruction, K = 16 per step) into a 128 x 512 fp32
// accumulator that fills TMEM.  Causal truncation: a tile only multiplies the N = (m0 + 128)/S columns it can see.
//
// The per-row top-k is the real cost (plain ALU).  4 x PF_NP epilogue warps: the PF_NP warps that share a TMEM lane
// quadrant hold the same 32 query rows and split each row's 32-column chunks between them (chunk c -> part c % PF_NP),
// combining per-row partial results through shared memory behind a named barrier.  Per row, all in registers except a
// <= 24-entry boundary list:
//   pass 0   row min / max
//   search   over equal-width value buckets of [min, max]: count(s >= t) per pass, 7 one-threshold passes over 128 buckets
//            (4 three-threshold passes over 256 buckets in the replicated mode below)
//   collect  the elements of the boundary bucket (value, id); the parts rank them by (value desc, id asc) between them:
//            the k-th is the threshold T, with id_T the last id taken among its equals
//   count    selected elements per chunk;  emit  ids with s > T or (s == T and id <= id_T) at the chunk's offset of the
//            row's output in global memory
// Columns beyond a row's causal candidates read as -inf, so the passes compare values only.  A row whose boundary
// bucket holds more than 24 elements (heavy ties) takes an exact bitwise radix search over order-preserving keys in
// part 0 alone (33 passes; warp-uniform because tcgen05.ld is warp-collective), which hands (T, id_T) to the others.
// Chunk-sized calls run the replicated mode (32-row tiles, 16 threads per row, one 32-column chunk per thread): row_topk_repl
// keeps the chunk in registers, searches on an fp16 image of it and exchanges through shared-memory atomics.
// Scores never leave the SM.  a7' loops the same MMA over the G heads of the group, turns each head's accumulator
// into softmax probabilities (two TMEM passes) summed into an L2-resident per-CTA scratch tile, and runs the same
// selection on that tile.
#include <cuda_fp16.h>

#include "sparda_internal.cuh"

#ifdef SPARDA_TRACE
__device__ unsigned long long* g_pf_trace;   // [gridDim.x][32] globaltimer stamps of warp 2 lane 0 (debug builds only)
extern "C" void sparda_debug_set_pf_trace(unsigned long long* p) { cudaMemcpyToSymbol(g_pf_trace, &p, sizeof(p)); }
#define PF_TRACE(i)                                                                           \
    if (threadIdx.x == 64) {                                                                  \
        unsigned long long t__;                                                               \
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t__));                               \
        g_pf_trace[blockIdx.x * 32 + (i)] = t__;                                              \
    }
#else
#define PF_TRACE(i)
#endif

namespace {

using namespace sparda;

#ifndef PF_NP_V
#define PF_NP_V 4
#endif
constexpr int PF_NP = PF_NP_V;    // epilogue warps per TMEM lane quadrant: the threads that share a query row
constexpr int PF_THREADS = 64 + 128 * PF_NP;   // warp 0: TMA producer, warp 1: TMEM owner + MMA issuer, then 4 * PF_NP epilogue warps
constexpr int PF_ROWS = 128;      // UMMA M
constexpr int PF_MAXN = 512;      // TMEM columns = max pooled keys per group
constexpr int PF_CAP = 24;        // boundary-list capacity per row
constexpr int PF_LIST_WORDS = 2 * PF_CAP;
constexpr int PF_WSTRIDE = 129;   // words between a thread's consecutive private words (bank-conflict free)
constexpr int PF_MAXK = 64;       // ids staged per row
constexpr int PF_BUCKET_BITS = 7;

template <int D>
struct PfSmem {
    static constexpr int KH = D / 64;                            // 64-element (128 B) K slabs
    static constexpr int B_SLAB = PF_MAXN * 128;                 // one K slab of B: 512 rows x 128 B
    static constexpr int A_SLAB = PF_ROWS * 128;
    static constexpr int OFF_B = 0;
    static constexpr int OFF_A = OFF_B + KH * B_SLAB;
    static constexpr int OFF_LIST = OFF_A + KH * A_SLAB;
    static constexpr int OFF_STAT = OFF_LIST + PF_LIST_WORDS * PF_WSTRIDE * 4;   // a7': (m, 1/l) per row, 1 KB
    static constexpr int OFF_COMB = OFF_STAT + PF_ROWS * 8;                   // exchange cells: [2][PF_NP][rows] float2
    static constexpr int OFF_NLIST = OFF_COMB + 2 * PF_NP * PF_ROWS * 8;      // boundary-list length per row
    static constexpr int OFF_CCNT = OFF_NLIST + PF_ROWS * 4;                  // selected count per (chunk, row), u8
    static constexpr int OFF_BAR = (OFF_CCNT + (PF_MAXN / 32) * PF_ROWS + 7) & ~7;
    static constexpr int OFF_CELL = (OFF_BAR + 64 + 15) & ~15;                // replicated mode: [PF_NCELL][32 rows] u32 exchange cells
    static constexpr int OFF_CNT16 = OFF_CELL + 8 * 32 * 4;                   // replicated mode: [32 rows][16 chunks] selected counts, u8
    static constexpr int OFF_STAGE = OFF_CNT16 + 32 * 16;                     // replicated mode: [32 rows][65] ids on their way out
    static constexpr int TOTAL = OFF_STAGE + 32 * 65 * 4 + 1024; // + slack for 1024-byte alignment
};

struct PfParams {
    int32_t* ids;        // [Hkv][n_rows][topk]
    float* scratch;      // a7': [gridDim.x][512][128] fp32 (column-major tile: scratch[j][row])
    int T, n_blocks, row0, n_rows, topk, Hkv, G;
    int mt_lo, n_tiles;  // absolute 128-row tiles covering [row0, row0 + n_rows)
    float scale_log2;    // a7': log2(e) / sqrt(D)
};

// ---- tcgen05 / TMEM helpers (inline PTX) ------------------------------------------------------------------------
__device__ __forceinline__ void tmem_alloc(uint32_t* smem_dst, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_dst)), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// mbarrier wait for a role that waits long (a whole epilogue): back off between polls so the spinning warp does not
// take issue slots from the warps that work
__device__ __forceinline__ void mbar_wait_backoff(uint64_t* bar, uint32_t parity, unsigned ns) {
    for (;;) {
        uint32_t ok;
        asm volatile(
            "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
        if (ok) break;
        __nanosleep(ns);
    }
}
// D[tmem] (+)= A[smem desc] * B[smem desc], bf16 x bf16 -> fp32, issued by one thread
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
        "}" ::"r"(tmem_d),
        "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
        : "memory");
}
// K-major operand tile in shared memory, rows of 128 B (64 bf16), 128-byte swizzle: 8-row atoms 1024 B apart
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr) {
    uint64_t d = (uint64_t)((smem_addr & 0x3FFFFu) >> 4);   // start address, 16-byte units
    d |= (uint64_t)(1024u >> 4) << 32;                        // stride byte offset between 8-row groups
    d |= (uint64_t)1 << 46;                                   // descriptor version (sm_100)
    d |= (uint64_t)2 << 61;                                   // SWIZZLE_128B
    return d;
}
// instruction descriptor: A, B bf16 K-major, D fp32, M = 128, N = n
__device__ __forceinline__ uint32_t umma_idesc(int n) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(PF_ROWS >> 4) << 24);
}
// this warp's 32 TMEM lanes x 32 consecutive fp32 columns -> one row of 32 values per thread
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32]) {
    uint32_t r[32];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n"
        "tcgen05.wait::ld.sync.aligned;"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
          "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]),
          "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}

// ---- where a row's scores come from: TMEM (a7) or the per-CTA scratch tile in global memory (a7') -----------------
struct TmemRow {
    uint32_t taddr;  // tmem base + (quadrant * 32) << 16
    __device__ __forceinline__ void load(int c, float (&v)[32]) const { tmem_ld32(taddr + c * 32, v); }
};
struct ScratchRow {
    const float* base;  // scratch + row; element j at base[j * PF_ROWS]
    __device__ __forceinline__ void load(int c, float (&v)[32]) const {
#pragma unroll
        for (int e = 0; e < 32; ++e) v[e] = __ldcg(base + (size_t)(c * 32 + e) * PF_ROWS);
    }
};

__device__ __forceinline__ float key_to_float(uint32_t key) {
    return __uint_as_float(key ^ ((key >> 31) ? 0x80000000u : 0xFFFFFFFFu));
}

// ---- the PF_NP epilogue warps that share a TMEM lane quadrant (same 32 query rows) split a row's 32-column chunks
// between them (chunk c belongs to part c % PF_NP) and combine per-row partial results through shared memory:
// write own partial, named barrier of the quadrant's PF_NP warps, read all parts.  Two buffers alternate, so one
// barrier per exchange is enough.
template <int NP>
struct PartComm {
    float2* comb;       // this row's cell of part 0, buffer 0; part stride PF_ROWS / (NP / PF_NP), see cell()
    int part, bar_id, buf;
    // cells: [2 buffers][NP parts][PF_ROWS * PF_NP / NP rows]: 4 parts x 128 rows, or 16 parts x 32 rows (replicated tile)
    static constexpr int ROWS = PF_ROWS * PF_NP / NP;
    __device__ __forceinline__ void sync() const { asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "n"(NP * 32) : "memory"); }
    __device__ __forceinline__ void put(float2 v) {
        buf ^= 1;
        comb[(buf * NP + part) * ROWS] = v;
        sync();
    }
    __device__ __forceinline__ float2 get(int p) const { return comb[(buf * NP + p) * ROWS]; }
    __device__ __forceinline__ int sum_int(int a) {
        put(make_float2(__int_as_float(a), 0.f));
        int s = 0;
#pragma unroll
        for (int p = 0; p < NP; ++p) s += __float_as_int(get(p).x);
        return s;
    }
};

// Exact per-row top-k of src[0 .. ncand) for the PF_NP threads that own one query row (one per part); the whole quadrant
// group calls it together (loads are warp-collective, exchanges are group barriers); a thread with active == false
// only keeps the others company.  The row's k ids are written to dst in ascending order.
template <int BPP, class Src, int NP>
__device__ __forceinline__ void row_topk(const Src& src, int ncand, int nch, int k, bool active, PartComm<NP>& pc,
                                         uint32_t* list /* row's list, stride PF_WSTRIDE */, uint32_t* n_list /* row's counter */,
                                         uint8_t* chunk_cnt /* row's [16] chunk counts, stride PF_ROWS */, int32_t* dst /* row's k ids in global memory */) {
    float v[32];
    const float NEG = -INFINITY;
    const int part = pc.part;
    if (!active) ncand = 0;
    if (part == 0) *n_list = 0;                       // ordered before the collection by the exchanges below
    // columns beyond the row's candidates read as -inf (only the last chunk of a warp's rows can hold any), so the
    // passes below compare values only: no index test per element
    auto load = [&](int c, float (&x)[32]) {
        src.load(c, x);
        if (__any_sync(0xffffffffu, c * 32 + 32 > ncand)) {
#pragma unroll
            for (int e = 0; e < 32; ++e) x[e] = c * 32 + e < ncand ? x[e] : NEG;
        }
    };
    // ---- pass 0: min / max over the candidates
    float lo = INFINITY, hi = -INFINITY;
    for (int c = part; c < nch; c += NP) {
        src.load(c, v);
#pragma unroll
        for (int e = 0; e < 32; ++e)
            if (c * 32 + e < ncand) { lo = fminf(lo, v[e]); hi = fmaxf(hi, v[e]); }
    }
    pc.put(make_float2(lo, hi));
#pragma unroll
    for (int p = 0; p < NP; ++p) { const float2 o = pc.get(p); lo = fminf(lo, o.x); hi = fmaxf(hi, o.y); }
    PF_TRACE(2);
    // ---- bucket search over 2^PF_BUCKET_BITS equal-width buckets of [min, max]: the largest bucket edge t_b with
    // count(s >= t_b) >= k.  BPP bits per pass: one threshold per pass (7 passes) when a thread holds several chunks, three
    // thresholds per pass (4 passes) in the replicated mode, where a pass is one chunk and mostly exchange latency.
    // Counts are accumulated as floats (FSET + FADD; exact up to 2^24).
    constexpr int NBITS = BPP == 2 ? 8 : PF_BUCKET_BITS;
    const float w = (hi - lo) * (1.0f / (1 << NBITS));
    int blo = 0, bhi = 1 << NBITS;                    // count(s >= t_blo) >= k > count(s >= t_bhi);  t_top = +inf
    int c_lo = ncand, c_hi = 0;
#pragma unroll 1
    for (int step = 0; step < NBITS / BPP; ++step) {
        if (BPP == 1) {
            const int mid = (blo + bhi) >> 1;
            const float t = fmaf((float)mid, w, lo);
            float cnt0 = 0.f, cnt1 = 0.f;
            for (int c = part; c < nch; c += NP) {
                load(c, v);
#pragma unroll
                for (int e = 0; e < 32; e += 2) {
                    cnt0 += v[e] >= t ? 1.0f : 0.0f;
                    cnt1 += v[e + 1] >= t ? 1.0f : 0.0f;
                }
            }
            const int cnt = pc.sum_int((int)(cnt0 + cnt1));
            if (cnt >= k) { blo = mid; c_lo = cnt; } else { bhi = mid; c_hi = cnt; }
        } else {
            const int q = (bhi - blo) >> 2;
            const float t1 = fmaf((float)(blo + q), w, lo), t2 = fmaf((float)(blo + 2 * q), w, lo), t3 = fmaf((float)(blo + 3 * q), w, lo);
            float n1 = 0.f, n2 = 0.f, n3 = 0.f;
            for (int c = part; c < nch; c += NP) {
                load(c, v);
#pragma unroll
                for (int e = 0; e < 32; ++e) {
                    n1 += v[e] >= t1 ? 1.0f : 0.0f;
                    n2 += v[e] >= t2 ? 1.0f : 0.0f;
                    n3 += v[e] >= t3 ? 1.0f : 0.0f;
                }
            }
            // three counts <= 512 each in one word: the sum over the parts cannot carry between the 10-bit fields
            const int packed = pc.sum_int((int)n1 | ((int)n2 << 10) | ((int)n3 << 20));
            const int c1 = packed & 1023, c2 = (packed >> 10) & 1023, c3 = (packed >> 20) & 1023;
            if (c3 >= k) { blo += 3 * q; c_lo = c3; }
            else if (c2 >= k) { blo += 2 * q; bhi = blo + q; c_lo = c2; c_hi = c3; }
            else if (c1 >= k) { blo += q; bhi = blo + q; c_lo = c1; c_hi = c2; }
            else { bhi = blo + q; c_hi = c1; }
        }
        PF_TRACE(3 + step);
    }
    const float tlo = fmaf((float)blo, w, lo);
    const float thi = bhi == (1 << NBITS) ? INFINITY : fmaf((float)bhi, w, lo);
    const int need = k - c_hi;                        // how many of the boundary bucket are selected (>= 1)
    const int n_b = c_lo - c_hi;                      // population of the boundary bucket
    const bool slow = active && (n_b > PF_CAP);
    float T = NEG;                                    // k-th largest value
    int jT = -1;                                      // selected among s == T: ids <= jT
    // ---- collect the boundary bucket (any order; entries carry their id) and resolve it exactly
    for (int c = part; c < nch; c += NP) {
        load(c, v);
#pragma unroll
        for (int e = 0; e < 32; ++e) {
            const int j = c * 32 + e;
            if (v[e] >= tlo && v[e] < thi && !slow) {
                const uint32_t n = atomicAdd(n_list, 1u);
                if (n < PF_CAP) {
                    list[(2 * n) * PF_WSTRIDE] = __float_as_uint(v[e]);
                    list[(2 * n + 1) * PF_WSTRIDE] = (uint32_t)j;
                }
            }
        }
    }
    pc.sync();
    PF_TRACE(10);
    {
        // the need-th largest of the list by (value desc, id asc): part p ranks the members e = p, p + NP, ... (their
        // ranks are distinct, so exactly one part finds the k-th) and the finder hands (T, jT) to the others
        float Tm = NEG;
        int jm = -1;
        if (active && !slow) {
            for (int e = part; e < n_b; e += NP) {
                const float se = __uint_as_float(list[(2 * e) * PF_WSTRIDE]);
                const int je = (int)list[(2 * e + 1) * PF_WSTRIDE];
                int rank = 0;
                int f = 0;
                for (; f + 4 <= n_b; f += 4) {       // four independent loads in flight
                    float sf[4];
                    int jf[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        sf[u] = __uint_as_float(list[(2 * (f + u)) * PF_WSTRIDE]);
                        jf[u] = (int)list[(2 * (f + u) + 1) * PF_WSTRIDE];
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) rank += (sf[u] > se || (sf[u] == se && jf[u] < je)) ? 1 : 0;
                }
                for (; f < n_b; ++f) {
                    const float sf = __uint_as_float(list[(2 * f) * PF_WSTRIDE]);
                    const int jf = (int)list[(2 * f + 1) * PF_WSTRIDE];
                    rank += (sf > se || (sf == se && jf < je)) ? 1 : 0;
                }
                if (rank == need - 1) { Tm = se; jm = je; }
            }
        }
        pc.put(make_float2(Tm, __int_as_float(jm)));
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const float2 o = pc.get(p);
            if (__float_as_int(o.y) >= 0) { T = o.x; jT = __float_as_int(o.y); }
        }
    }
    // ---- heavy ties (rare): part 0 alone searches the k-th largest order-preserving key bit by bit over all chunks, finds
    // the id of the last equal it takes, and hands (T, jT) to the other parts.  Warp-uniform, and the same in every warp
    // of the quadrant (they hold the same rows).
    if (__any_sync(0xffffffffu, slow)) {
        if (part == 0) {
            uint32_t tk = 0;
#pragma unroll 1
            for (int bit = 31; bit >= 0; --bit) {
                const uint32_t cand = tk | (1u << bit);
                int cnt = 0;
                for (int c = 0; c < nch; ++c) {
                    load(c, v);
#pragma unroll
                    for (int e = 0; e < 32; ++e) cnt += (c * 32 + e < ncand && orderable(v[e] + 0.0f) >= cand) ? 1 : 0;
                }
                if (cnt >= k) tk = cand;
            }
            int cgt = 0;
            for (int c = 0; c < nch; ++c) {
                load(c, v);
#pragma unroll
                for (int e = 0; e < 32; ++e) cgt += (c * 32 + e < ncand && orderable(v[e] + 0.0f) > tk) ? 1 : 0;
            }
            int eq_left = k - cgt, j_last = -1;       // take the first k - cgt equals in ascending id
            for (int c = 0; c < nch; ++c) {
                load(c, v);
#pragma unroll
                for (int e = 0; e < 32; ++e)
                    if (c * 32 + e < ncand && orderable(v[e] + 0.0f) == tk && eq_left > 0) { j_last = c * 32 + e; --eq_left; }
            }
            if (slow) { T = key_to_float(tk); jT = j_last; }
        }
        pc.put(make_float2(T, __int_as_float(jT)));
        if (slow) { const float2 o = pc.get(0); T = o.x; jT = __float_as_int(o.y); }
    }
    PF_TRACE(11);
    // ---- selected element: s > T, or s == T with id <= jT (+-0 compare equal, as in the oracle's ordering).  Count per
    // chunk, exchange, then every chunk writes its ids at its offset of the row's output: ascending ids.
    for (int c = part; c < nch; c += NP) {
        load(c, v);
        int n = 0;
#pragma unroll
        for (int e = 0; e < 32; ++e) {
            const int j = c * 32 + e;
            n += (v[e] > T || (v[e] == T && j <= jT)) ? 1 : 0;
        }
        chunk_cnt[c * PF_ROWS] = (uint8_t)n;
    }
    pc.sync();
    PF_TRACE(12);
    for (int c = part; c < nch; c += NP) {
        int pos = 0;
#pragma unroll
        for (int cc = 0; cc < PF_MAXN / 32; ++cc) {     // independent loads; chunks at or beyond nch are never read as < c
            const int n = cc < c ? (int)chunk_cnt[cc * PF_ROWS] : 0;
            pos += n;
        }
        load(c, v);
#pragma unroll
        for (int e = 0; e < 32; ++e) {
            const int j = c * 32 + e;
            if ((v[e] > T || (v[e] == T && j <= jT)) && pos < k) dst[pos++] = j;
        }
    }
}

// ---- replicated mode (chunk launches): 16 threads per query row, ONE 32-column chunk per thread.  The chunk is read from
// TMEM once and stays in registers; the bucket search runs on a monotone fp16 image of it, two elements per instruction
// (HSET2 + HADD2); the 16 parts of a row combine their partial results by shared-memory atomics on one cell per (exchange,
// row) -- lanes of a warp hit 32 different cells, so an exchange is one conflict-free atomic per warp, one CTA barrier and
// one load per thread instead of one store and 16 loads.  Same result as row_topk: the k largest by (value desc, id asc),
// ids ascending.  Any monotone bucket map keeps the selection exact: an element of a higher bucket is larger than every
// element of a lower one, and the boundary bucket is ranked on the fp32 values.
constexpr int PF_NCELL = 8;                 // 0 min, 1 max, 2..5 search steps, 6 T, 7 id_T
constexpr int PF_SSTRIDE = PF_MAXK + 1;     // words per row of the shared-memory output tile (odd: rows fall into different banks)
__device__ __forceinline__ uint32_t pf_cell_init(int i) { return i == 0 ? 0xFFFFFFFFu : i == 6 ? 0xFF800000u /* -inf */ : i == 7 ? 0xFFFFFFFFu /* -1 */ : 0u; }

template <class Src>
__device__ __forceinline__ void row_topk_repl(const Src& src, int ncand, int nch, int k, bool active, int part,
                                              uint32_t* cell /* this row's column of the [PF_NCELL][32] cells */,
                                              uint8_t* cnt16 /* this row's 16 chunk counts, 16-byte aligned */,
                                              uint32_t* list /* row's list, stride PF_WSTRIDE */, uint32_t* n_list,
                                              int32_t* stage_row /* this row's k ids in the shared-memory output tile */) {
    constexpr int NP = 16;
    const float NEG = -INFINITY;
    auto sync = [] { asm volatile("bar.sync 1, 512;" ::: "memory"); };
    if (!active) ncand = 0;
    const bool has = part < nch;            // warp-uniform (the parts are warps)
    const int base = part * 32;
    float v[32];
    bool ragged = false;                    // the chunk reaches beyond some row's candidates (warp-uniform)
    // ---- the chunk, once; columns beyond the row's candidates read as -inf; row min / max over the candidates
    float lo = INFINITY, hi = NEG;
    if (has) {
        src.load(part, v);
        ragged = __any_sync(0xffffffffu, base + 32 > ncand);
        if (ragged) {
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                const bool ok = base + e < ncand;
                lo = fminf(lo, ok ? v[e] : INFINITY);
                v[e] = ok ? v[e] : NEG;
                hi = fmaxf(hi, v[e]);
            }
        } else {
#pragma unroll
            for (int e = 0; e < 32; ++e) { lo = fminf(lo, v[e]); hi = fmaxf(hi, v[e]); }
        }
        if (base < ncand) {
            atomicMin(cell + 0 * 32, orderable(lo + 0.0f));
            atomicMax(cell + 1 * 32, orderable(hi + 0.0f));
        }
    }
    sync();
    PF_TRACE(2);
    lo = key_to_float(cell[0 * 32]);
    hi = key_to_float(cell[1 * 32]);
    // ---- fp16 image: x = (v - lo) * 256 / (hi - lo) in [0, 256], -1 beyond the candidates; bucket b = [b, b + 1)
    const float scale = hi > lo ? __fdividef(256.0f, hi - lo) : 0.f;   // any scale keeps the bucket map monotone
    const float off = -lo * scale;
    __half2 h[16];
    if (has && !ragged) {
#pragma unroll
        for (int w = 0; w < 16; ++w)
            h[w] = __floats2half2_rn(fmaxf(fmaf(v[2 * w], scale, off), 0.f), fmaxf(fmaf(v[2 * w + 1], scale, off), 0.f));
    } else if (has) {
#pragma unroll
        for (int w = 0; w < 16; ++w) {
            const float x0 = v[2 * w] == NEG ? -1.f : fmaxf(fmaf(v[2 * w], scale, off), 0.f);
            const float x1 = v[2 * w + 1] == NEG ? -1.f : fmaxf(fmaf(v[2 * w + 1], scale, off), 0.f);
            h[w] = __floats2half2_rn(x0, x1);
        }
    } else {
#pragma unroll
        for (int w = 0; w < 16; ++w) h[w] = __float2half2_rn(-1.f);
    }
    // ---- bucket search, three thresholds per step over 256 buckets: the largest bucket edge t with count(x >= t) >= k
    int blo = 0, bhi = 256;                 // count(x >= blo) >= k > count(x >= bhi)
    int c_lo = ncand, c_hi = 0;
#pragma unroll 1
    for (int step = 0; step < 4; ++step) {
        const int q = (bhi - blo) >> 2;
        const __half2 t1 = __float2half2_rn((float)(blo + q)), t2 = __float2half2_rn((float)(blo + 2 * q)), t3 = __float2half2_rn((float)(blo + 3 * q));
        __half2 a1 = __float2half2_rn(0.f), a2 = a1, a3 = a1;
#pragma unroll
        for (int w = 0; w < 16; ++w) {
            a1 = __hadd2(a1, __hge2(h[w], t1));
            a2 = __hadd2(a2, __hge2(h[w], t2));
            a3 = __hadd2(a3, __hge2(h[w], t3));
        }
        if (has) {
            const int n1 = (int)(__low2float(a1) + __high2float(a1)), n2 = (int)(__low2float(a2) + __high2float(a2)),
                      n3 = (int)(__low2float(a3) + __high2float(a3));
            // three counts <= 512 each in one word: the sum over the parts cannot carry between the 10-bit fields
            atomicAdd(cell + (2 + step) * 32, (uint32_t)(n1 | (n2 << 10) | (n3 << 20)));
        }
        sync();
        const int packed = (int)cell[(2 + step) * 32];
        const int c1 = packed & 1023, c2 = (packed >> 10) & 1023, c3 = (packed >> 20) & 1023;
        if (c3 >= k) { blo += 3 * q; c_lo = c3; }
        else if (c2 >= k) { blo += 2 * q; bhi = blo + q; c_lo = c2; c_hi = c3; }
        else if (c1 >= k) { blo += q; bhi = blo + q; c_lo = c1; c_hi = c2; }
        else { bhi = blo + q; c_hi = c1; }
        PF_TRACE(3 + step);
    }
    const int need = k - c_hi;              // how many of the boundary bucket are selected (>= 1)
    const int n_b = c_lo - c_hi;            // population of the boundary bucket
    const bool slow = active && (n_b > PF_CAP);
    const bool any_slow = __any_sync(0xffffffffu, slow);   // the same in every warp: they hold the same rows
    // ---- elements above the boundary bucket, per chunk: with the selected members of the boundary list they give every
    // chunk's offset in the row's output without another exchange
    {
        int above = 0;
        if (has && bhi < 256) {
            const __half2 tb = __float2half2_rn((float)bhi);
            __half2 a = __float2half2_rn(0.f);
#pragma unroll
            for (int w = 0; w < 16; ++w) a = __hadd2(a, __hge2(h[w], tb));
            above = (int)(__low2float(a) + __high2float(a));
        }
        cnt16[part] = (uint8_t)above;
    }
    // ---- collect the boundary bucket [blo, bhi) (any order; entries carry their fp32 value and id): a bit per element, one
    // atomic per thread for its slots in the row's list, then the (few) set bits are written out
    if (has) {
        const __half2 hb = __float2half2_rn((float)blo), hb1 = __float2half2_rn(bhi == 256 ? INFINITY : (float)bhi);
        uint32_t bits = 0;
#pragma unroll
        for (int w = 0; w < 16; ++w) {
            const unsigned m = __hge2_mask(h[w], hb) & __hlt2_mask(h[w], hb1);
            bits |= ((m & 1u) | ((m >> 15) & 2u)) << (2 * w);
        }
        if (bits != 0u && !slow) {          // not slow: the bucket's n_b <= PF_CAP members all fit
            uint32_t* slot = list + 2 * PF_WSTRIDE * atomicAdd(n_list, (uint32_t)__popc(bits));
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                if ((bits >> e) & 1u) {
                    slot[0] = __float_as_uint(v[e]);
                    slot[PF_WSTRIDE] = (uint32_t)(base + e);
                    slot += 2 * PF_WSTRIDE;
                }
            }
        }
    }
    sync();
    PF_TRACE(10);
    if (part == 0) {                        // the min / max / search cells have been read by everybody: re-arm them for the next tile
#pragma unroll
        for (int i = 0; i < 6; ++i) cell[i * 32] = pf_cell_init(i);
    }
    // ---- the need-th largest of the list by (value desc, id asc): part p ranks the members p, p + 16, ...; exactly one
    // finds it and publishes (T, id_T)
    if (active && !slow) {
        for (int e = part; e < n_b; e += NP) {
            const float se = __uint_as_float(list[(2 * e) * PF_WSTRIDE]);
            const int je = (int)list[(2 * e + 1) * PF_WSTRIDE];
            int rank = 0;
            int f = 0;
            for (; f + 4 <= n_b; f += 4) {           // four independent loads in flight
                float sf[4];
                int jf[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    sf[u] = __uint_as_float(list[(2 * (f + u)) * PF_WSTRIDE]);
                    jf[u] = (int)list[(2 * (f + u) + 1) * PF_WSTRIDE];
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) rank += (sf[u] > se || (sf[u] == se && jf[u] < je)) ? 1 : 0;
            }
            for (; f < n_b; ++f) {
                const float sf = __uint_as_float(list[(2 * f) * PF_WSTRIDE]);
                const int jf = (int)list[(2 * f + 1) * PF_WSTRIDE];
                rank += (sf > se || (sf == se && jf < je)) ? 1 : 0;
            }
            if (rank == need - 1) { cell[6 * 32] = __float_as_uint(se); cell[7 * 32] = (uint32_t)je; }
        }
    }
    // ---- heavy ties (rare): part 0 alone searches the k-th largest order-preserving key bit by bit over all chunks and
    // finds the id of the last equal it takes.  Warp-uniform, and the same in every warp (they hold the same rows).
    if (any_slow) {
        if (part == 0) {
            float u[32];
            uint32_t tk = 0;
#pragma unroll 1
            for (int bit = 31; bit >= 0; --bit) {
                const uint32_t cand = tk | (1u << bit);
                int cnt = 0;
                for (int c = 0; c < nch; ++c) {
                    src.load(c, u);
#pragma unroll
                    for (int e = 0; e < 32; ++e) cnt += (c * 32 + e < ncand && orderable(u[e] + 0.0f) >= cand) ? 1 : 0;
                }
                if (cnt >= k) tk = cand;
            }
            int cgt = 0;
            for (int c = 0; c < nch; ++c) {
                src.load(c, u);
#pragma unroll
                for (int e = 0; e < 32; ++e) cgt += (c * 32 + e < ncand && orderable(u[e] + 0.0f) > tk) ? 1 : 0;
            }
            int eq_left = k - cgt, j_last = -1;       // take the first k - cgt equals in ascending id
            for (int c = 0; c < nch; ++c) {
                src.load(c, u);
#pragma unroll
                for (int e = 0; e < 32; ++e)
                    if (c * 32 + e < ncand && orderable(u[e] + 0.0f) == tk && eq_left > 0) { j_last = c * 32 + e; --eq_left; }
            }
            if (slow) { cell[6 * 32] = __float_as_uint(key_to_float(tk)); cell[7 * 32] = (uint32_t)j_last; }
        }
    }
    sync();
    PF_TRACE(11);
    const float T = __uint_as_float(cell[6 * 32]);    // k-th largest value (-inf: nothing to select)
    const int jT = (int)cell[7 * 32];                 // selected among s == T: ids <= jT
    // ---- selected element: s > T, or s == T with id <= jT.  Every chunk writes its ids at its offset of the row's k slots
    // in a shared-memory tile (row stride 65 words: the 32 rows of a warp fall into different banks), ascending ids; the
    // tile then leaves in coalesced stores.  Offset of chunk p = elements above the boundary bucket in the chunks before it
    // + selected members of the boundary list with smaller ids.
    const int eT = jT - base;               // elements e <= eT of this chunk equal to T are selected
    if (any_slow) {                         // a row of the tile resolved heavy ties without a list: exchange exact counts (rare)
        int n = 0;
        if (has) {
#pragma unroll
            for (int e = 0; e < 32; ++e) n += (v[e] > T || (v[e] == T && e <= eT)) ? 1 : 0;
        }
        cnt16[part] = (uint8_t)n;
        sync();
    }
    if (has) {
        const uint4 c4 = *reinterpret_cast<const uint4*>(cnt16);
        const uint32_t cw[4] = {c4.x, c4.y, c4.z, c4.w};
        unsigned upos = 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {       // bytes of the chunks before this one
            const int nb = min(max(part - 4 * i, 0), 4);
            const uint32_t mask = nb >= 4 ? 0xFFFFFFFFu : ((1u << (8 * nb)) - 1u);
            upos = __dp4a(cw[i] & mask, 0x01010101u, upos);
        }
        if (!any_slow && active) {
            for (int f0 = 0; f0 < n_b; f0 += 4) {     // four independent pairs of loads in flight; entries >= n_b are never counted
                float sf[4];
                int jf[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int f = min(f0 + u, PF_CAP - 1);
                    sf[u] = __uint_as_float(list[(2 * f) * PF_WSTRIDE]);
                    jf[u] = (int)list[(2 * f + 1) * PF_WSTRIDE];
                }
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    upos += (f0 + u < n_b && jf[u] < base && (sf[u] > T || (sf[u] == T && jf[u] <= jT))) ? 1u : 0u;
            }
        }
        PF_TRACE(14);
        int32_t* out = stage_row + (int)upos;
#pragma unroll
        for (int e = 0; e < 32; ++e) {
            if (v[e] > T || (v[e] == T && e <= eT)) *out++ = base + e;
        }
    }
    PF_TRACE(15);
}

// REPL (chunk launches with few tiles): a CTA owns 32 query rows instead of 128.  Its A tile holds the same 32 rows four
// times (four 32-row TMA boxes), so the four TMEM lane quadrants carry four copies of the rows' scores and ALL 16 epilogue
// warps work on those 32 rows, 16 threads per row (chunk c -> part c % 16).  The contraction is done four times over --
// it is ~1 % of the kernel -- and a 2048-row chunk spreads over 128 CTAs instead of 32.
template <int D, bool BASELINE, bool REPL>
__global__ void __launch_bounds__(PF_THREADS, 1)
prefill_select_kernel(const __grid_constant__ CUtensorMap tmapA, const __grid_constant__ CUtensorMap tmapB, PfParams p) {
    constexpr int TROWS = REPL ? 32 : PF_ROWS;        // query rows per tile
    constexpr int NP = REPL ? 4 * PF_NP : PF_NP;      // threads per query row
    static_assert(!REPL || PF_NP == 4, "the replicated mode spreads a row over 16 epilogue warps");
    using SM = PfSmem<D>;
    constexpr int KH = SM::KH;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + SM::OFF_BAR);
    uint64_t* b_full = bars + 0;
    uint64_t* a_full = bars + 1;
    uint64_t* a_empty = bars + 2;
    uint64_t* mma_done = bars + 3;
    uint64_t* tmem_empty = bars + 4;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 5);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = blockIdx.x % p.Hkv;                 // this CTA's group: its Kpool stays resident
    const int cta = blockIdx.x / p.Hkv;
    const int n_cta = gridDim.x / p.Hkv;              // CTAs per group
    const int NH = BASELINE ? p.G : 1;                // A-operand passes per tile (heads of the group)

    if (tid == 0) {
        mbar_init(b_full, 1);
        mbar_init(a_full, 1);
        mbar_init(a_empty, 1);
        mbar_init(mma_done, 1);
        mbar_init(tmem_empty, 4 * PF_NP);
        mbar_fence_init();
        fence_proxy_async_smem();
        tma_prefetch_desc(&tmapA);
        tma_prefetch_desc(&tmapB);
    }
    if (warp == 1) tmem_alloc(tmem_slot, PF_MAXN);
    if (REPL) {   // exchange cells of row_topk_repl, armed for the first tile (the function re-arms them for the next)
        uint32_t* cells = reinterpret_cast<uint32_t*>(smem + SM::OFF_CELL);
        for (int i = tid; i < PF_NCELL * 32; i += PF_THREADS) cells[i] = pf_cell_init(i >> 5);
        if (tid < 32) reinterpret_cast<uint32_t*>(smem + SM::OFF_NLIST)[tid] = 0;
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    PF_TRACE(0);
    // Programmatic dependent launch: the prologue above and the load of the group's pooled keys (never written by a kernel
    // that signals completion early, see sparda.h cfg.no_pdl) overlap the previous kernel's tail; the Forecast / query tiles
    // and every store (ids, the comparison selector's scratch tile) wait for it.
    pdl_launch_dependents();

    // Tile schedule (identical in every role): tiles sorted by cost (descending row index), dealt in a snake over the
    // group's CTAs.  Tile s covers rows [m0, m0 + 128), m0 = (mt_lo + n_tiles - 1 - s) * 128.
    auto tile_of_round = [&](int r) -> int {
        const int s = r * n_cta + ((r & 1) ? (n_cta - 1 - cta) : cta);
        return s < p.n_tiles ? (p.mt_lo + p.n_tiles - 1 - s) : -1;
    };
    const int n_rounds = (p.n_tiles + n_cta - 1) / n_cta;
    auto tile_ncols = [&](int mt) -> int { return min(p.n_blocks, (mt * TROWS + TROWS) / 64); };  // visible blocks of the tile's last row

    // replicated mode: the tile's ids leave the shared-memory tile in coalesced stores (the ranked rows only; the others are
    // filled directly).  Called by all 16 epilogue warps.
    auto repl_store_tile = [&](const int32_t* stage, const PfParams& pp, int grp, int mt) {
        asm volatile("bar.sync 1, 512;" ::: "memory");
        PF_TRACE(16);
        if (tid - 64 < 32) {                // everybody has read (T, id_T) and the list: re-arm them for the next tile
            uint32_t* cells = reinterpret_cast<uint32_t*>(smem + SM::OFF_CELL) + (tid - 64);
            cells[6 * 32] = pf_cell_init(6);
            cells[7 * 32] = pf_cell_init(7);
            reinterpret_cast<uint32_t*>(smem + SM::OFF_NLIST)[tid - 64] = 0;
        }
        const int row = (tid - 64) >> 4, c0 = (tid - 64) & 15;   // 16 threads per row, 64-byte runs
        const int i = mt * 32 + row;
        if (i >= pp.row0 && i < pp.row0 + pp.n_rows && min(pp.n_blocks, (i + 1) / 64) > pp.topk) {
            int32_t* drow = pp.ids + ((size_t)grp * pp.n_rows + (i - pp.row0)) * pp.topk;
            for (int c = c0; c < pp.topk; c += 16) drow[c] = stage[row * PF_SSTRIDE + c];
        }
    };

    if (warp == 0) {
        // =============================== TMA producer ===============================
        if (lane == 0) {
            // causal truncation of the B operand too: this CTA's tiles see at most the columns of its first (highest) tile
            const int mt0 = tile_of_round(0);
            const int nb_boxes = mt0 < 0 ? 1 : (tile_ncols(mt0) + 255) / 256;
            mbar_arrive_expect_tx(b_full, (uint32_t)(KH * nb_boxes * 256 * 128));
            for (int kh = 0; kh < KH; ++kh)
                for (int nh = 0; nh < nb_boxes; ++nh)
                    tma_load_2d(smem + SM::OFF_B + kh * SM::B_SLAB + nh * 256 * 128, &tmapB, kh * 64, g * p.n_blocks + nh * 256, b_full);
            pdl_wait();
            uint32_t it = 0;
            for (int r = 0; r < n_rounds; ++r) {
                const int mt = tile_of_round(r);
                if (mt < 0 || tile_ncols(mt) <= p.topk) continue;   // nothing to rank: every candidate is selected
                for (int h = 0; h < NH; ++h, ++it) {
                    mbar_wait_backoff(a_empty, (it & 1) ^ 1, 400);
                    mbar_arrive_expect_tx(a_full, (uint32_t)(KH * SM::A_SLAB));
                    const int arow = (BASELINE ? (g * p.G + h) : g) * p.T + mt * TROWS;
                    for (int kh = 0; kh < KH; ++kh)
                        for (int rg = 0; rg < PF_ROWS / TROWS; ++rg)   // REPL: the same 32 rows into all four row groups
                            tma_load_2d(smem + SM::OFF_A + kh * SM::A_SLAB + rg * TROWS * 128, &tmapA, kh * 64, arow, a_full);
                }
            }
        }
    } else if (warp == 1) {
        // =============================== MMA issuer ===============================
        if (lane == 0) {
            mbar_wait(b_full, 0);
            const uint32_t a_addr = smem_u32(smem + SM::OFF_A), b_addr = smem_u32(smem + SM::OFF_B);
            uint32_t it = 0;
            for (int r = 0; r < n_rounds; ++r) {
                const int mt = tile_of_round(r);
                if (mt < 0 || tile_ncols(mt) <= p.topk) continue;
                const int ncols = (tile_ncols(mt) + 15) & ~15;
                for (int h = 0; h < NH; ++h, ++it) {
                    mbar_wait_backoff(a_full, it & 1, 100);
                    mbar_wait_backoff(tmem_empty, (it & 1) ^ 1, 200);
                    tc_fence_after();
                    for (int nh = 0; nh * 256 < ncols; ++nh) {
                        const int n = min(256, ncols - nh * 256);
                        const uint32_t idesc = umma_idesc(n);
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks) {
                            const uint64_t da = umma_desc_sw128(a_addr + (ks >> 2) * SM::A_SLAB + (ks & 3) * 32);
                            const uint64_t db = umma_desc_sw128(b_addr + (ks >> 2) * SM::B_SLAB + nh * 256 * 128 + (ks & 3) * 32);
                            umma_bf16(tmem_base + nh * 256, da, db, idesc, ks > 0 ? 1u : 0u);
                        }
                    }
                    tc_commit(a_empty);    // A tile may be overwritten once these MMAs have read it
                    tc_commit(mma_done);   // accumulator complete
                }
            }
        }
    } else {
        // =============================== epilogue: PF_NP threads per query row ===============================
        pdl_wait();
        const int q = warp & 3;                                  // TMEM lane quadrant this warp may access
        const int part = REPL ? q * PF_NP + ((warp - 2) >> 2) : (warp - 2) >> 2;   // which share of the row's chunks this warp takes
        const int trow = REPL ? lane : q * 32 + lane;            // row within the tile
        uint32_t* list = reinterpret_cast<uint32_t*>(smem + SM::OFF_LIST) + trow;
        uint32_t* n_list = reinterpret_cast<uint32_t*>(smem + SM::OFF_NLIST) + trow;
        uint8_t* chunk_cnt = smem + SM::OFF_CCNT + trow;
        PartComm<NP> pc{reinterpret_cast<float2*>(smem + SM::OFF_COMB) + trow, part, REPL ? 1 : 1 + q, 0};
        float* scr = BASELINE ? p.scratch + (size_t)blockIdx.x * PF_MAXN * PF_ROWS + trow : nullptr;
        const TmemRow trsrc{tmem_base + ((uint32_t)(q * 32) << 16)};
        uint32_t it = 0;
        for (int r = 0; r < n_rounds; ++r) {
            const int mt = tile_of_round(r);
            if (mt < 0) continue;
            const int i = mt * TROWS + trow;                      // query position of this thread
            const bool in_chunk = i >= p.row0 && i < p.row0 + p.n_rows;
            const int ncand = min(p.n_blocks, (i + 1) / 64);
            int32_t* dst = p.ids + ((size_t)g * p.n_rows + (i - p.row0)) * p.topk;
            const int ncols = tile_ncols(mt);
            // this part's share of the row's k output positions
            const int s_lo = min(p.topk, part * ((p.topk + NP - 1) / NP)), s_hi = min(p.topk, s_lo + (p.topk + NP - 1) / NP);
            if (ncols <= p.topk) {                               // whole tile: every candidate is selected (reading q5)
                if (in_chunk)
                    for (int s = s_lo; s < s_hi; ++s) dst[s] = s < ncand ? s : -1;
                continue;
            }
            const int wmax = min(p.n_blocks, (mt * TROWS + (REPL ? 0 : q * 32) + 32) / 64);   // candidates of the warp's last row
            const int nch = (wmax + 31) / 32;
            const bool ranked = in_chunk && ncand > p.topk;
            if (BASELINE) {
                // a7': per head, softmax over the causal candidates of the row, summed into the scratch tile
                float v[32];
                for (int h = 0; h < NH; ++h, ++it) {
                    mbar_wait_backoff(mma_done, it & 1, 100);
                    tc_fence_after();
                    float m = -INFINITY;
                    for (int c = part; c < nch; c += NP) {
                        trsrc.load(c, v);
#pragma unroll
                        for (int e = 0; e < 32; ++e)
                            if (c * 32 + e < ncand) m = fmaxf(m, v[e]);
                    }
                    pc.put(make_float2(m, 0.f));
#pragma unroll
                    for (int pp = 0; pp < NP; ++pp) m = fmaxf(m, pc.get(pp).x);
                    const float ms = m * p.scale_log2;
                    float l = 0.f;
                    for (int c = part; c < nch; c += NP) {
                        trsrc.load(c, v);
#pragma unroll
                        for (int e = 0; e < 32; ++e)
                            if (c * 32 + e < ncand) l += exp2f(fmaf(v[e], p.scale_log2, -ms));
                    }
                    pc.put(make_float2(l, 0.f));
                    l = 0.f;
#pragma unroll
                    for (int pp = 0; pp < NP; ++pp) l += pc.get(pp).x;   // same order in every part
                    const float inv = ncand > 0 ? 1.0f / l : 0.f;
                    for (int c = part; c < nch; c += NP) {
                        trsrc.load(c, v);
#pragma unroll
                        for (int e = 0; e < 32; ++e) {
                            const int j = c * 32 + e;
                            if (j < ncand) {
                                const float pr = exp2f(fmaf(v[e], p.scale_log2, -ms)) * inv;
                                float* a = scr + (size_t)j * PF_ROWS;
                                __stcg(a, h == 0 ? pr : __ldcg(a) + pr);
                            }
                        }
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(tmem_empty);
                }
                if (__any_sync(0xffffffffu, ranked)) {
                    if constexpr (REPL) {
                        int32_t* stage = reinterpret_cast<int32_t*>(smem + SM::OFF_STAGE);
                        row_topk_repl(ScratchRow{scr}, ncand, nch, p.topk, ranked, part, reinterpret_cast<uint32_t*>(smem + SM::OFF_CELL) + trow,
                                      smem + SM::OFF_CNT16 + trow * 16, list, n_list, stage + trow * PF_SSTRIDE);
                        repl_store_tile(stage, p, g, mt);
                    } else
                        row_topk<1>(ScratchRow{scr}, ncand, nch, p.topk, ranked, pc, list, n_list, chunk_cnt, dst);
                }
            } else {
                mbar_wait_backoff(mma_done, it & 1, 100);
                ++it;
                tc_fence_after();
                PF_TRACE(1);
                if (__any_sync(0xffffffffu, ranked)) {
                    if constexpr (REPL) {
                        int32_t* stage = reinterpret_cast<int32_t*>(smem + SM::OFF_STAGE);
                        row_topk_repl(trsrc, ncand, nch, p.topk, ranked, part, reinterpret_cast<uint32_t*>(smem + SM::OFF_CELL) + trow,
                                      smem + SM::OFF_CNT16 + trow * 16, list, n_list, stage + trow * PF_SSTRIDE);
                        repl_store_tile(stage, p, g, mt);
                    } else
                        row_topk<1>(trsrc, ncand, nch, p.topk, ranked, pc, list, n_list, chunk_cnt, dst);
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tmem_empty);
            }
            if (!ranked && in_chunk) {
                for (int s = s_lo; s < s_hi; ++s) dst[s] = s < ncand ? s : -1;
            }
            PF_TRACE(13);
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, PF_MAXN);
    }
}

template <int D, bool BASELINE, bool REPL>
int launch_mode(sparda_ctx* ctx, const void* A, const void* Kpool, int T, int n_blocks, int row0, int n_rows, int topk, int32_t* ids,
                cudaStream_t st) {
    using SM = PfSmem<D>;
    constexpr int TROWS = REPL ? 32 : PF_ROWS;
    const int Hkv = ctx->cfg.n_kv_heads, G = ctx->G;
    CUtensorMap mapA, mapB;   // copies: a later lookup can never change a descriptor held here
    int rc = sparda_get_tmap(ctx, A, (uint64_t)(BASELINE ? Hkv * G : Hkv) * T, D, TROWS, &mapA);
    if (rc) return rc;
    rc = sparda_get_tmap(ctx, Kpool, (uint64_t)Hkv * n_blocks, D, 256, &mapB);
    if (rc) return rc;
    int per_group = ctx->sm_count / Hkv;
    if (per_group < 1) return SPARDA_EINVAL;
    PfParams p;
    p.ids = ids;
    p.T = T;
    p.n_blocks = n_blocks;
    p.row0 = row0;
    p.n_rows = n_rows;
    p.topk = topk;
    p.Hkv = Hkv;
    p.G = G;
    p.mt_lo = row0 / TROWS;
    p.n_tiles = (row0 + n_rows + TROWS - 1) / TROWS - p.mt_lo;
    if (per_group > p.n_tiles) per_group = p.n_tiles;
    p.scale_log2 = 1.4426950408889634f / sqrtf((float)D);
    p.scratch = nullptr;
    if (BASELINE) p.scratch = ctx->pf_scratch;
    sparda_kernel_state& ks = ctx->kstate[SPARDA_K_PF_0 + (D == 128 ? 4 : 0) + (BASELINE ? 2 : 0) + (REPL ? 1 : 0)];
    if (!ks.attr_set) {
        SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(prefill_select_kernel<D, BASELINE, REPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM::TOTAL));
        ks.attr_set = true;
    }
    cudaLaunchAttribute at[1] = {sparda_pdl_attr()};
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((unsigned)(per_group * Hkv), 1, 1);
    lc.blockDim = dim3(PF_THREADS, 1, 1);
    lc.dynamicSmemBytes = SM::TOTAL;
    lc.stream = st;
    lc.attrs = at;
    lc.numAttrs = sparda_use_pdl(ctx) ? 1 : 0;
    SPARDA_CUDA_TRY(ctx, cudaLaunchKernelEx(&lc, prefill_select_kernel<D, BASELINE, REPL>, mapA, mapB, p));
    SPARDA_CUDA_TRY(ctx, cudaGetLastError());
    ctx->launches++;
    return SPARDA_OK;
}

// A call whose 128-row tiles would leave a quarter of the SMs or more idle (a 2048-row chunk is 16 tiles per group) runs in
// the replicated mode: 32-row tiles, 16 threads per row (measured break-even: about one 128-row tile per SM).
template <int D, bool BASELINE>
int launch(sparda_ctx* ctx, const void* A, const void* Kpool, int T, int n_blocks, int row0, int n_rows, int topk, int32_t* ids,
           cudaStream_t st) {
    const int tiles128 = (row0 + n_rows + PF_ROWS - 1) / PF_ROWS - row0 / PF_ROWS;
    if (PF_NP == 4 && 4 * tiles128 * ctx->cfg.n_kv_heads <= 3 * ctx->sm_count)
        return launch_mode<D, BASELINE, true>(ctx, A, Kpool, T, n_blocks, row0, n_rows, topk, ids, st);
    return launch_mode<D, BASELINE, false>(ctx, A, Kpool, T, n_blocks, row0, n_rows, topk, ids, st);
}

}  // namespace

// Supported range of the tcgen05 path: Nb <= 512 pooled keys per group (one 128 x 512 fp32 accumulator = all of TMEM),
// topk <= 64, D in {64, 128}.  [BJ] configs[4]: T = 32768, Nb = 512, k = 64.
int sparda_launch_prefill_select(sparda_ctx* ctx, const void* F, const void* Kpool, int T, int n_blocks, int row0, int n_rows,
                                 int topk, int32_t* ids, cudaStream_t st) {
    if (n_blocks > PF_MAXN || topk > PF_MAXK) return SPARDA_EINVAL;
    return ctx->cfg.head_dim == 128 ? launch<128, false>(ctx, F, Kpool, T, n_blocks, row0, n_rows, topk, ids, st)
                                    : launch<64, false>(ctx, F, Kpool, T, n_blocks, row0, n_rows, topk, ids, st);
}
int sparda_launch_prefill_baseline(sparda_ctx* ctx, const void* Q, const void* Kpool, int T, int n_blocks, int row0, int n_rows,
                                   int topk, int32_t* ids, cudaStream_t st) {
    if (n_blocks > PF_MAXN || topk > PF_MAXK) return SPARDA_EINVAL;
    return ctx->cfg.head_dim == 128 ? launch<128, true>(ctx, Q, Kpool, T, n_blocks, row0, n_rows, topk, ids, st)
                                    : launch<64, true>(ctx, Q, Kpool, T, n_blocks, row0, n_rows, topk, ids, st);
}
