// Block-sparse GQA decode attention on the 5th-generation tensor cores: the "swap-AB" form, Eq.5.
//
// An EXPERIMENT behind cfg.attn_impl = 1 (the mma.sync kernel of sparse_decode.cu stays the default; DESIGN.md 5.3 has the
// measured comparison).  tcgen05.mma needs M >= 64, and a decode step has only G <= 16 query heads per group, so the tokens
// take the M side:
//     S^T [128 tokens x 16 heads] = K [128 x D] . Q^T [D x 16]          A = the K tile as TMA delivers it (K-major, SW128)
//     O^T [D = 128 x 16 heads]   += V^T [D x 128 tokens] . P [128 x 16]  A = the V tile as TMA delivers it, read MN-major
// Two 64-token blocks (pool slots) per iteration.  Accumulators live in TMEM (32 columns); one token per thread in the
// softmax: thread t of the 128 reads its row of S^T (tcgen05.ld), the per-head block max is a redux.sync per head and one
// exchange between the four warps, P goes to shared memory as the K-major B operand of the second product, and the running
// row sums stay in registers until the end.  When a head's maximum grows, the O^T accumulator is rescaled in TMEM
// (tcgen05.ld -> multiply -> tcgen05.st).  A fifth warp feeds a ring of 64 KiB stages with TMA and owns the TMEM allocation.
// The CTA's partial (m, l, O) then takes the same ways out as in sparse_decode.cu: stored directly (one CTA per row) or
// reduced inside a thread-block cluster through distributed shared memory (2, 4 or 8 CTAs per row).
// Supported: D = 128, G <= 16, row-aligned splits; everything else stays on the mma.sync kernel.
#include "sparda_internal.cuh"

#ifdef SPARDA_TRACE
__device__ unsigned long long* g_t5_trace;   // [gridDim.x][8] cycles per phase, summed over the iterations of thread 0 (debug builds only)
extern "C" void sparda_debug_set_t5_trace(unsigned long long* p) { cudaMemcpyToSymbol(g_t5_trace, &p, sizeof(p)); }
#define T5_T(i) if (tid == 0) { const long long n__ = clock64(); tr_[i] += n__ - tl_; tl_ = n__; }
#else
#define T5_T(i)
#endif

namespace {

using namespace sparda;

constexpr int T5_THREADS = 160;                 // 4 softmax warps (one token per thread) + 1 producer warp
constexpr int T5_STAGES = 3;
constexpr int T5_STAGE_BYTES = 65536;           // K: [d 0-63: block a | block b][d 64-127: a | b], then V the same
constexpr int T5_OFF_Q = T5_STAGES * T5_STAGE_BYTES;          // Q: 2 slabs of [16 heads][128 B]
constexpr int T5_OFF_P = T5_OFF_Q + 4096;                      // P^T: 2 buffers x 2 slabs of [16 heads][128 B]
constexpr int T5_OFF_X = T5_OFF_P + 8192;                      // partial O [16][132] fp32, then the cluster landing area
constexpr int T5_OROW = 132;
constexpr int T5_TOTAL = T5_OFF_X + 16 * T5_OROW * 4 + 16 * 128 * 4 + 16 * 2 * 4 + 1024;

struct T5Params {
    const int32_t* ids;
    __nv_bfloat16* O;
    int topk, indexed, n_slots, Hq, Hkv, G;
    int per_cta;           // slots per CTA (divides topk)
    float scale_log2;
};

__device__ __forceinline__ void t5_tmem_alloc(uint32_t* smem_dst, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_dst)), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void t5_tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void t5_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void t5_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void t5_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void t5_mma(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}" ::"r"(tmem_d),
        "l"(da), "l"(db), "r"(idesc), "r"(acc)
        : "memory");
}
// shared-memory matrix descriptor, 128-byte swizzle, 8-row groups 1024 B apart; lbo: distance between 64-element groups along
// the MN dimension of an MN-major operand (unused for a K-major one)
__device__ __forceinline__ uint64_t t5_desc(uint32_t addr, uint32_t lbo_bytes) {
    uint64_t d = (uint64_t)((addr & 0x3FFFFu) >> 4);
    d |= (uint64_t)(lbo_bytes >> 4) << 16;
    d |= (uint64_t)(1024u >> 4) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}
// instruction descriptor: bf16 x bf16 -> fp32, M = 128, N = 16; a_mn = 1: A is MN-major
__device__ __forceinline__ uint32_t t5_idesc(int a_mn) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_mn << 15) | ((16u >> 3) << 17) | ((128u >> 4) << 24);
}
__device__ __forceinline__ void t5_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n"
        "tcgen05.wait::ld.sync.aligned;"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void t5_st16(uint32_t taddr, const float (&v)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};\n"
        "tcgen05.wait::st.sync.aligned;" ::"r"(taddr),
        "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])),
        "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7])),
        "r"(__float_as_uint(v[8])), "r"(__float_as_uint(v[9])), "r"(__float_as_uint(v[10])), "r"(__float_as_uint(v[11])),
        "r"(__float_as_uint(v[12])), "r"(__float_as_uint(v[13])), "r"(__float_as_uint(v[14])), "r"(__float_as_uint(v[15]))
        : "memory");
}
// order-preserving float <-> int (for redux.sync.max on floats)
__device__ __forceinline__ int f2ord(float f) { const int b = __float_as_int(f); return b >= 0 ? b : b ^ 0x7FFFFFFF; }
__device__ __forceinline__ float ord2f(int o) { return __int_as_float(o >= 0 ? o : o ^ 0x7FFFFFFF); }
__device__ __forceinline__ void softmax_sync() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

template <bool CL>
__global__ void __launch_bounds__(T5_THREADS, 1)
sparse_decode_tc5_kernel(const __grid_constant__ CUtensorMap tmapKV, const __grid_constant__ CUtensorMap tmapQ, T5Params p) {
    constexpr int D = 128;
    extern __shared__ uint8_t t5_raw[];
    __shared__ uint64_t full_k[T5_STAGES], full_v[T5_STAGES], empty[T5_STAGES], bar_q, bar_s, bar_o[2];   // bar_o[j & 1]: P V product of iteration j
    __shared__ uint32_t tmem_slot;
    __shared__ int s_max[2][4][16];        // per (buffer, warp, head): block maximum (ordered ints)
    __shared__ float s_l[4][16];
    uint8_t* smem = t5_raw + ((1024u - (smem_u32(t5_raw) & 1023u)) & 1023u);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int s_per = p.topk / p.per_cta;                 // CTAs per row
    const int r = blockIdx.x / s_per, part = blockIdx.x % s_per;
    const int slot0 = part * p.per_cta;
    const int n_iter = (p.per_cta + 1) / 2;
    const int32_t* ids_row = p.ids + (size_t)r * p.topk;
    const int b = r / p.Hkv, g = r % p.Hkv;

    if (tid == 0) {
        for (int i = 0; i < T5_STAGES; ++i) { mbar_init(&full_k[i], 1); mbar_init(&full_v[i], 1); mbar_init(&empty[i], 1); }
        mbar_init(&bar_q, 1); mbar_init(&bar_s, 1); mbar_init(&bar_o[0], 1); mbar_init(&bar_o[1], 1);
        mbar_fence_init();
        fence_proxy_async_smem();
        tma_prefetch_desc(&tmapKV);
        tma_prefetch_desc(&tmapQ);
    }
    if (w == 4) t5_tmem_alloc(&tmem_slot, 32);
    t5_fence_before();
    __syncthreads();
    t5_fence_after();
    const uint32_t tmem = tmem_slot;
    pdl_wait();
    pdl_launch_dependents();

    // first valid slot of this CTA's range: the stand-in source for padded (-1) slots, whose pool contents are undefined
    int sub = -1;
    for (int s = 0; s < p.per_cta; ++s)
        if (__ldg(ids_row + slot0 + s) >= 0) { sub = s; break; }
    auto src_row = [&](int s, int plane) -> int {         // first row of slot s's K (plane 0) or V (plane 1) tile in the tensor map
        int sl = slot0 + s;
        const int id = __ldg(ids_row + sl);
        if (id < 0) sl = slot0 + sub;
        const int idx = p.indexed ? max(__ldg(ids_row + sl), 0) : sl;
        return ((r * p.n_slots + idx) * 2 + plane) * 64;
    };

    float l_run[16];
#pragma unroll
    for (int h = 0; h < 16; ++h) l_run[h] = 0.f;
    float m_run[16];
#pragma unroll
    for (int h = 0; h < 16; ++h) m_run[h] = -INFINITY;

    if (sub >= 0) {
        if (w == 4) {
            // =============================== producer: Q once, then the ring of K / V pairs ===============================
            if (lane == 0) {
                mbar_arrive_expect_tx(&bar_q, 4096);
                tma_load_2d(smem + T5_OFF_Q, &tmapQ, 0, b * p.Hq + g * p.G, &bar_q);
                tma_load_2d(smem + T5_OFF_Q + 2048, &tmapQ, 64, b * p.Hq + g * p.G, &bar_q);
                for (int i = 0; i < n_iter; ++i) {
                    const int st = i % T5_STAGES;
                    if (i >= T5_STAGES) mbar_wait(&empty[st], ((i / T5_STAGES) - 1) & 1);
                    uint8_t* base = smem + (size_t)st * T5_STAGE_BYTES;
                    const int sa = 2 * i, sb = min(2 * i + 1, p.per_cta - 1);    // an odd tail repeats its last slot (masked below)
                    mbar_arrive_expect_tx(&full_k[st], 32768);
                    tma_load_2d(base, &tmapKV, 0, src_row(sa, 0), &full_k[st]);
                    tma_load_2d(base + 8192, &tmapKV, 0, src_row(sb, 0), &full_k[st]);
                    tma_load_2d(base + 16384, &tmapKV, 64, src_row(sa, 0), &full_k[st]);
                    tma_load_2d(base + 24576, &tmapKV, 64, src_row(sb, 0), &full_k[st]);
                    mbar_arrive_expect_tx(&full_v[st], 32768);
                    tma_load_2d(base + 32768, &tmapKV, 0, src_row(sa, 1), &full_v[st]);
                    tma_load_2d(base + 32768 + 8192, &tmapKV, 0, src_row(sb, 1), &full_v[st]);
                    tma_load_2d(base + 32768 + 16384, &tmapKV, 64, src_row(sa, 1), &full_v[st]);
                    tma_load_2d(base + 32768 + 24576, &tmapKV, 64, src_row(sb, 1), &full_v[st]);
                }
            }
        } else {
            // =============================== 128 softmax threads; thread 0 also issues the MMAs ===============================
            const uint32_t t_s = tmem + ((uint32_t)(w * 32) << 16);            // S^T: columns 0-15 of this warp's lanes
            const uint32_t t_o = t_s + 16;                                     // O^T: columns 16-31
            const uint32_t q_addr = smem_u32(smem + T5_OFF_Q);
            const uint32_t id_s = t5_idesc(0), id_o = t5_idesc(1);
            bool o_started = false;
            // S^T = K . Q^T of iteration i (8 k-steps of 16 elements of d), issued by thread 0 one iteration ahead: as soon as
            // every thread holds S(i-1) in registers the single S buffer is free, and the product overlaps that softmax
            auto issue_s = [&](int i) {
                const int st = i % T5_STAGES;
                const uint32_t kbase = smem_u32(smem + (size_t)st * T5_STAGE_BYTES);
                mbar_wait(&full_k[st], (i / T5_STAGES) & 1);
                t5_fence_after();
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks)
                    t5_mma(tmem, t5_desc(kbase + (ks >> 2) * 16384 + (ks & 3) * 32, 0), t5_desc(q_addr + (ks >> 2) * 2048 + (ks & 3) * 32, 0), id_s,
                           ks > 0 ? 1u : 0u);
                t5_commit(&bar_s);
            };
            if (tid == 0) {
                mbar_wait(&bar_q, 0);
                issue_s(0);
            }
#ifdef SPARDA_TRACE
            long long tr_[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tl_ = clock64();
#endif
            for (int i = 0; i < n_iter; ++i) {
                const int st = i % T5_STAGES;
                const uint32_t ph = (i / T5_STAGES) & 1;
                const uint32_t vbase = smem_u32(smem + (size_t)st * T5_STAGE_BYTES) + 32768;
                const uint32_t pbase = smem_u32(smem + T5_OFF_P + (i & 1) * 4096);
                mbar_wait(&bar_s, i & 1);
                T5_T(0);
                t5_fence_after();
                float s[16];
                t5_ld16(t_s, s);
                t5_fence_before();
                T5_T(1);
                // token of this thread: slot 2i (threads 0-63) or 2i+1 (threads 64-127); padded and repeated slots are masked
                const int my_slot = 2 * i + (tid >> 6);
                const bool live = my_slot < p.per_cta && __ldg(ids_row + slot0 + my_slot) >= 0;
                // ---- block maximum per head: redux over the warp, exchange between the four warps
#pragma unroll
                for (int h = 0; h < 16; ++h) {
                    const int o = __reduce_max_sync(0xffffffffu, live ? f2ord(s[h]) : f2ord(-INFINITY));
                    if (lane == 0) s_max[i & 1][w][h] = o;
                }
                softmax_sync();
                T5_T(2);
                if (tid == 0 && i + 1 < n_iter) issue_s(i + 1);
                __syncwarp();
                T5_T(3);
                float resc[16];
                bool grow = false;
#pragma unroll
                for (int h = 0; h < 16; ++h) {
                    const int o = max(max(s_max[i & 1][0][h], s_max[i & 1][1][h]), max(s_max[i & 1][2][h], s_max[i & 1][3][h]));
                    const float mb = ord2f(o) * p.scale_log2;
                    const float mn = fmaxf(m_run[h], mb);
                    resc[h] = (mn == -INFINITY) ? 1.f : exp2f(m_run[h] - mn);
                    grow |= mn > m_run[h];
                    m_run[h] = mn;
                }
                // ---- a maximum grew: rescale the accumulator where it lives (uniform over the CTA: every thread sees the same maxima)
                if (grow && o_started) {
                    mbar_wait(&bar_o[(i - 1) & 1], ((i - 1) >> 1) & 1);   // the previous P V product has completed
                    t5_fence_after();
                    float o[16];
                    t5_ld16(t_o, o);
#pragma unroll
                    for (int h = 0; h < 16; ++h) o[h] *= resc[h];
                    t5_st16(t_o, o);
                }
#pragma unroll
                for (int h = 0; h < 16; ++h) l_run[h] *= resc[h];
                // ---- P = exp2(s * scale - m), rounded to bf16 (the rounded weights also feed the row sums), into the K-major B tile
                T5_T(4);
                if (i >= 2) mbar_wait(&bar_o[i & 1], ((i - 2) >> 1) & 1);   // the product that read this P buffer (iteration i-2) has completed
                const int tok = tid & 63, slab = tid >> 6;
#pragma unroll
                for (int h = 0; h < 16; ++h) {
                    const float pf = live && m_run[h] > -INFINITY ? exp2f(fmaf(s[h], p.scale_log2, -m_run[h])) : 0.f;
                    const __nv_bfloat16 pb = __float2bfloat16_rn(pf);
                    l_run[h] += __bfloat162float(pb);
                    const uint32_t off = slab * 2048 + (h >> 3) * 1024 + (h & 7) * 128 + (((tok >> 3) ^ (h & 7)) << 4) + (tok & 7) * 2;
                    asm volatile("st.shared.u16 [%0], %1;" ::"r"(pbase + off), "h"(__bfloat16_as_ushort(pb)) : "memory");
                }
                T5_T(5);
                fence_proxy_async_smem();
                t5_fence_before();
                softmax_sync();
                T5_T(6);
                // ---- O^T += V^T . P  (8 k-steps of 16 tokens); the commit also hands the stage back to the producer
                if (tid == 0) {
                    mbar_wait(&full_v[st], ph);
                    t5_fence_after();
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks)
                        t5_mma(tmem + 16, t5_desc(vbase + ks * 2048, 16384), t5_desc(pbase + (ks >> 2) * 2048 + (ks & 3) * 32, 0), id_o,
                               (o_started || ks > 0) ? 1u : 0u);
                    t5_commit(&bar_o[i & 1]);
                    t5_commit(&empty[st]);
                }
                __syncwarp();
                o_started = true;
                T5_T(7);
            }
#ifdef SPARDA_TRACE
            if (tid == 0 && g_t5_trace)
                for (int q = 0; q < 8; ++q) g_t5_trace[blockIdx.x * 8 + q] = (unsigned long long)tr_[q];
#endif
            // ---- the CTA's partial: O^T row d of this thread -> exchange buffer [head][d]; row sums across the 128 threads
            mbar_wait(&bar_o[(n_iter - 1) & 1], ((n_iter - 1) >> 1) & 1);
            t5_fence_after();
            float o[16];
            t5_ld16(t_o, o);
            float* xo = reinterpret_cast<float*>(smem + T5_OFF_X);
#pragma unroll
            for (int h = 0; h < 16; ++h) xo[h * T5_OROW + tid] = o[h];
#pragma unroll
            for (int h = 0; h < 16; ++h) {
                float v = l_run[h];
#pragma unroll
                for (int off = 16; off >= 1; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
                if (lane == 0) s_l[w][h] = v;
            }
        }
    }
    t5_fence_before();
    __syncthreads();
    // ---- (m, l, O) of this CTA is in shared memory (or empty: sub < 0).  One CTA per row: normalise and store; else: cluster.
    float* xo = reinterpret_cast<float*>(smem + T5_OFF_X);
    __nv_bfloat16* obase = p.O + (size_t)(b * p.Hq + g * p.G) * D;
    if (!CL) {
        for (int it = tid; it < p.G * (D / 4); it += T5_THREADS) {
            const int row = it / (D / 4), c4 = it % (D / 4);
            const float L = sub >= 0 ? s_l[0][row] + s_l[1][row] + s_l[2][row] + s_l[3][row] : 0.f;
            const float inv = L > 0.f ? 1.f / L : 0.f;
            const float4 v = sub >= 0 ? *reinterpret_cast<const float4*>(xo + row * T5_OROW + c4 * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
            uint2 u;
            u.x = pack_bf16(v.x * inv, v.y * inv);
            u.y = pack_bf16(v.z * inv, v.w * inv);
            *reinterpret_cast<uint2*>(obase + (size_t)row * D + c4 * 4) = u;
        }
    } else {
        // as in sparse_decode.cu: every CTA sends each head row's partial (m, l, O) to the CTA that owns that head row
        const int n = s_per, rows_per = 16 / n;
        float* land = xo + 16 * T5_OROW;
        float* land_ml = land + 16 * D;
        const uint32_t land_u32 = smem_u32(land), ml_u32 = smem_u32(land_ml);
        // the running maxima are identical in every softmax thread; thread 0 publishes them for this phase
        __shared__ float s_m[16];
        if (tid < 16) s_m[tid] = -INFINITY;
        __syncthreads();
        if (tid == 0 && sub >= 0)
            for (int h = 0; h < 16; ++h) s_m[h] = m_run[h];
        asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");   // landing areas are free, peers run
        for (int it = tid; it < 16 * (D / 4); it += T5_THREADS) {
            const int row = it / (D / 4), c4 = it % (D / 4);
            const float M = s_m[row];
            const float L = sub >= 0 ? s_l[0][row] + s_l[1][row] + s_l[2][row] + s_l[3][row] : 0.f;
            const float4 v = sub >= 0 ? *reinterpret_cast<const float4*>(xo + row * T5_OROW + c4 * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
            const uint32_t owner = (uint32_t)(row / rows_per), lrow = (uint32_t)(row % rows_per);
            uint32_t dst, dml;
            asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(dst) : "r"(land_u32 + ((part * rows_per + lrow) * D + c4 * 4) * 4), "r"(owner));
            asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(dst), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
            if (c4 == 0) {
                asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(dml) : "r"(ml_u32 + ((part * rows_per + lrow) * 2) * 4), "r"(owner));
                asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(dml), "f"(M), "f"(L) : "memory");
            }
        }
        asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
        for (int it = tid; it < rows_per * (D / 4); it += T5_THREADS) {
            const int lrow = it / (D / 4), c4 = it % (D / 4);
            const int row = part * rows_per + lrow;
            if (row >= p.G) continue;
            float M = -INFINITY;
            for (int q = 0; q < n; ++q) M = fmaxf(M, land_ml[(q * rows_per + lrow) * 2]);
            float L = 0.f;
            float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
            for (int q = 0; q < n; ++q) {
                const float wg = (M == -INFINITY) ? 0.f : exp2f(land_ml[(q * rows_per + lrow) * 2] - M);
                L += wg * land_ml[(q * rows_per + lrow) * 2 + 1];
                const float4 v = *reinterpret_cast<const float4*>(land + ((size_t)(q * rows_per + lrow) * D + c4 * 4));
                acc.x += wg * v.x; acc.y += wg * v.y; acc.z += wg * v.z; acc.w += wg * v.w;
            }
            const float inv = L > 0.f ? 1.f / L : 0.f;
            uint2 u;
            u.x = pack_bf16(acc.x * inv, acc.y * inv);
            u.y = pack_bf16(acc.z * inv, acc.w * inv);
            *reinterpret_cast<uint2*>(obase + (size_t)row * D + c4 * 4) = u;
        }
    }
    __syncthreads();
    if (w == 4) {
        t5_fence_after();
        t5_tmem_dealloc(tmem, 32);
    }
}

template <bool CL>
int t5_launch(sparda_ctx* ctx, const CUtensorMap& mkv, const CUtensorMap& mq, const T5Params& p, int C, int cluster, cudaStream_t st) {
    auto kern = sparse_decode_tc5_kernel<CL>;
    sparda_kernel_state& ks = ctx->kstate[CL ? SPARDA_K_ATTN_T5_CL : SPARDA_K_ATTN_T5];
    if (!ks.attr_set) {
        SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, T5_TOTAL));
        ks.attr_set = true;
    }
    cudaLaunchConfig_t lc = {};
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    at[1] = sparda_pdl_attr();
    lc.attrs = at;
    lc.numAttrs = 1;
    lc.gridDim = dim3((unsigned)C, 1, 1);
    lc.blockDim = dim3(T5_THREADS, 1, 1);
    lc.dynamicSmemBytes = T5_TOTAL;
    lc.stream = st;
    if (CL) {
        if (ks.max_clusters[cluster] == 0) {
            int n = 0;
            if (cudaOccupancyMaxActiveClusters(&n, kern, &lc) != cudaSuccess) n = -1;
            (void)cudaGetLastError();
            ks.max_clusters[cluster] = n > 0 ? n : -1;
        }
        if (ks.max_clusters[cluster] * cluster < C) return 1;
    }
    lc.numAttrs = sparda_use_pdl(ctx) ? 2 : 1;
    SPARDA_CUDA_TRY(ctx, cudaLaunchKernelEx(&lc, kern, mkv, mq, p));
    return SPARDA_OK;
}

}  // namespace

// Returns SPARDA_OK when the tcgen05 kernel took the launch, 1 when the shape is outside its range (the caller falls back to
// the mma.sync kernel), or an error.
int sparda_launch_attn_tc5(sparda_ctx* ctx, const void* Q, const void* pool, const int32_t* ids, int topk, int indexed, int n_slots,
                           void* O, cudaStream_t st) {
    if (ctx->cfg.head_dim != 128 || ctx->G > 16) return 1;
    const int C = sparda_resolve_attn_ctas(ctx, topk);
    if (C % ctx->R != 0) return 1;
    const int s_per = C / ctx->R;
    if (topk % s_per != 0 || !(s_per == 1 || s_per == 2 || s_per == 4 || s_per == 8)) return 1;
    CUtensorMap mkv, mq;
    int rc = sparda_get_tmap(ctx, pool, (uint64_t)ctx->R * n_slots * 2 * 64, 128, 64, &mkv);
    if (rc) return rc;
    rc = sparda_get_tmap(ctx, Q, (uint64_t)ctx->cfg.batch * ctx->cfg.n_q_heads, 128, 16, &mq);
    if (rc) return rc;
    T5Params p;
    p.ids = ids;
    p.O = (__nv_bfloat16*)O;
    p.topk = topk;
    p.indexed = indexed;
    p.n_slots = n_slots;
    p.Hq = ctx->cfg.n_q_heads;
    p.Hkv = ctx->cfg.n_kv_heads;
    p.G = ctx->G;
    p.per_cta = topk / s_per;
    p.scale_log2 = 1.4426950408889634f / sqrtf(128.0f);
    rc = s_per == 1 ? t5_launch<false>(ctx, mkv, mq, p, C, 1, st) : t5_launch<true>(ctx, mkv, mq, p, C, s_per, st);
    if (rc) return rc;
    ctx->last_attn_cluster = s_per == 1 ? 0 : s_per;
    ctx->launches++;
    return SPARDA_OK;
}
