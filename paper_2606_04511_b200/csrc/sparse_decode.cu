// Block-sparse GQA decode attention over the gathered blocks (a5) and over a device-resident cache
// addressed by block id (a6, layer 0).  Eq.5, Alg.2 l.7:
//   O_h = softmax_t( q_h . k_t / sqrt(D) ) V   over every token t of every selected block of row r = b*Hkv + h/G.
//
// Flat split-K flash-decode.  The R*k pool slots of the launch form one flat work list that is cut into
// gridDim.x equal contiguous ranges (grid = a multiple of the SM count, so there is no wave-quantisation tail);
// a CTA walks its range row segment by row segment.  NW consumer warps per CTA, each with its own
// shared-memory stage (one block's K and V tiles, 2*S*D*2 bytes).  Lane 0 of a warp stages the warp's next block
// with TMA tensor-map loads (cp.async.bulk.tensor.2d, 64x64 boxes, 128-byte swizzle so ldmatrix is bank-conflict
// free) completing on per-stage mbarriers (K and V separately: QK^T starts when K lands, and the next K load is
// issued as soon as QK^T has consumed the tile).  The group's G <= 16 query heads are the M = 16 rows of
// mma.sync.m16n8k16 (bf16 in, fp32 accumulate): S = Q K^T (16 x 64 per block), online softmax in the exp2
// domain, O += P V.  Warp partials (m, l, O) are merged through shared memory.  The CTA partials of one row are reduced
// inside a thread-block cluster through distributed shared memory when the split is row-aligned with 2, 4, 8 or 16 CTAs per
// row (the [BJ] shapes), else through an L2-resident workspace by the last CTA to finish that row (ticket).  One bf16
// rounding.
// HBM-bound by design: 16 FLOP per KV byte at G = 16; the tensor pipe idles most of the time.
#include "sparda_internal.cuh"

#ifdef SPARDA_TRACE
__device__ unsigned long long* g_trace;   // [gridDim.x][8] globaltimer stamps (debug builds only)
extern "C" void sparda_debug_set_trace(unsigned long long* p) { cudaMemcpyToSymbol(g_trace, &p, sizeof(p)); }
#define TRACE(i)                                                                              \
    if (threadIdx.x == 0) {                                                                   \
        unsigned long long t__;                                                               \
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t__));                               \
        g_trace[blockIdx.x * 8 + (i)] = t__;                                                  \
    }
#else
#define TRACE(i)
#endif

namespace {

using namespace sparda;

constexpr int S_BLK = 64;

template <int D, int NW>
struct AttnSmem {
    static constexpr int TILE_BYTES = S_BLK * D * 2;        // one K (or V) tile
    static constexpr int STAGE_BYTES = 2 * TILE_BYTES;      // K then V
    static constexpr int OROW = D + 4;                      // padded fp32 row of a warp partial
    static constexpr int XCHG_WARP = 16 * OROW * 4;         // one warp's partial O (16 heads x D fp32)
    static constexpr int OFF_XCHG = NW * STAGE_BYTES;       // exchange area: separate from the stages, so the next
                                                            // segment's tiles can be in flight during a merge
    static constexpr int TOTAL = OFF_XCHG + 2 * NW * XCHG_WARP + 1024;   // two exchange buffers + alignment slack
};

struct AttnParams {
    const uint32_t* Q;     // bf16 pairs
    const int32_t* ids;
    const int32_t* seq_len; // [R] tokens in the row's cache, or nullptr = every listed block is complete (sparda_sparse_decode_varlen)
    __nv_bfloat16* O;
    float* part_O;         // [R][max_splits][16][D]
    float* part_ml;        // [R][max_splits][2][16]
    unsigned int* tickets; // [R]
    int topk, indexed, n_slots, Hq, Hkv, G, max_splits;
    int W;                 // R * topk flat slots (< 2^31)
    int quota, rem;        // W = gridDim.x * quota + rem: CTA c owns quota + (c < rem) slots from c * quota + min(c, rem)
    float scale_log2;
};

// owner(f): the CTA whose flat range holds slot f (inverse of the map in AttnParams)
__device__ __forceinline__ int flat_owner(int f, int quota, int rem) {
    const int thr = rem * (quota + 1);
    return f < thr ? f / (quota + 1) : rem + (f - thr) / quota;
}

// CL (row-aligned splits, s = 2, 4, 8 or 16 CTAs per row launched as one cluster): the CTA partials of a row are reduced
// through distributed shared memory instead of the L2 workspace -- every CTA sends each head row's partial (m, l, O) to the
// CTA that owns that head row (16 / s rows each), one cluster barrier, every CTA normalises and stores its rows.  No ticket,
// no fence, no global round trip, and the final merge is spread over the cluster.
// VARLEN (sparda_sparse_decode_varlen): p.seq_len[r] tokens exist in row r's cache; the partly filled newest block is masked.  Its own
// instantiation: the D = 128 kernel sits at the 255-register limit and the extra live values must not cost the default path.
template <int D, int NW, int MINB, bool CL, bool VARLEN>
__global__ void __launch_bounds__(NW * 32, MINB) sparse_decode_kernel(const __grid_constant__ CUtensorMap tmap, AttnParams p) {
    using SM = AttnSmem<D, NW>;
    constexpr int NT = NW * 32;
    constexpr int KSTEPS = D / 16;  // k-steps of Q K^T
    constexpr int DT = D / 8;       // n-tiles of P V
    constexpr int HALVES = D / 64;  // 64-element TMA boxes per row
    extern __shared__ uint8_t smem_raw[];
    __shared__ uint64_t bar_k[NW], bar_v[NW];
    __shared__ float s_ml[1][NW][2][16];
    __shared__ unsigned int s_last;
    __shared__ uint64_t bar_m;
    __shared__ uint64_t bar_red;     // CL: completes when every CTA's partials of the head rows this CTA owns have landed (tx bytes)
    __shared__ __align__(128) float s_pm[16 * 32];
    __shared__ float s_w[16 * 16], s_run[16], s_resc[16], s_newmax[16];

    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int gid = lane >> 2, tig = lane & 3;

    TRACE(0);
    if (tid == 0) {
        for (int i = 0; i < NW; ++i) { mbar_init(&bar_k[i], 1); mbar_init(&bar_v[i], 1); }
        mbar_init(&bar_m, 1);
        if (CL) {
            // cluster reduction: this CTA owns 16 / n head rows and expects (m, l, O[D]) of each of them from each of the n CTAs
            mbar_init(&bar_red, 1);
            mbar_arrive_expect_tx(&bar_red, 16u * (D * 4 + 8));
        }
        mbar_fence_init();
        fence_proxy_async_smem();
        tma_prefetch_desc(&tmap);
    }
    __syncthreads();
    // CL: every CTA of the cluster is running, with bar_red armed, before anyone stores into a neighbour's shared memory:
    // arrive now, wait in front of the reduction (by then everybody has long arrived)
    if (CL) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    pdl_wait();                  // the prologue above overlaps the previous kernel's tail; global memory from here on
    pdl_launch_dependents();

    uint8_t* stage = smem + (size_t)w * SM::STAGE_BYTES;
    const uint32_t k_base = smem_u32(stage), v_base = k_base + SM::TILE_BYTES;
    uint32_t phase = 0;
    // per-lane ldmatrix row offsets (swizzle: 16-byte chunk index ^= row & 7; rows are 128 B inside a box)
    const int mi = lane >> 3, ri = lane & 7;

    const int f_begin = (int)blockIdx.x * p.quota + min((int)blockIdx.x, p.rem);
    const int f_end = f_begin + p.quota + ((int)blockIdx.x < p.rem ? 1 : 0);
    struct Seg { int r, s0, s1; };
    auto seg_at = [&](int f) -> Seg {   // the row segment that starts at flat slot f
        Seg t;
        t.r = f / p.topk;
        t.s0 = f - t.r * p.topk;
        t.s1 = min(p.topk, t.s0 + (f_end - f));
        return t;
    };
    // this warp's first item at or after flat position f: slot s0 + w of the first segment long enough to have one
    auto first_item = [&](int f, int& r_out, int& s_out) -> bool {
        while (f < f_end) {
            const Seg t = seg_at(f);
            if (t.s0 + w < t.s1) { r_out = t.r; s_out = t.s0 + w; return true; }
            f += t.s1 - t.s0;
        }
        return false;
    };
    // Tiles are staged whether or not the slot is valid (id -1 = padding, rare: fewer candidates than k); an invalid
    // slot is skipped after its tiles land.  This keeps the ids load off the path to the first TMA issue.
    auto tile_row = [&](int r, int slot, int plane) -> int {
        int idx = slot;
        if (p.indexed) idx = max(__ldg(p.ids + (size_t)r * p.topk + slot), 0);
        return (((r * p.n_slots + idx) * 2 + plane) * S_BLK);
    };
    auto issue_k = [&](int r, int slot) {
        mbar_arrive_expect_tx(&bar_k[w], SM::TILE_BYTES);
#pragma unroll
        for (int h = 0; h < HALVES; ++h) tma_load_2d(stage + h * 8192, &tmap, h * 64, tile_row(r, slot, 0), &bar_k[w]);
    };
    auto issue_v = [&](int r, int slot) {
        mbar_arrive_expect_tx(&bar_v[w], SM::TILE_BYTES);
#pragma unroll
        for (int h = 0; h < HALVES; ++h)
            tma_load_2d(stage + SM::TILE_BYTES + h * 8192, &tmap, h * 64, tile_row(r, slot, 1), &bar_v[w]);
    };

    // ---- CTA merge of the warp partials in exchange buffer `buf` (all threads; a CTA barrier precedes it): a whole-row
    // segment is normalised and stored, a partial-row segment goes to the row's slot `part` of the L2-resident workspace
    constexpr int C4 = D / 4;
    auto cta_merge = [&](int buf, int r, int part, int n_parts) {
        const int b = r / p.Hkv, g = r % p.Hkv;
        __nv_bfloat16* obase = p.O + (size_t)(b * p.Hq + g * p.G) * D;
        float* po = p.part_O + ((size_t)r * p.max_splits + part) * 16 * D;
        float* pml = p.part_ml + ((size_t)r * p.max_splits + part) * 32;
        for (int it = tid; it < 16 * C4; it += NT) {   // items = (head row, float4 column); rows >= G carry zeros
            const int row = it / C4, c4 = it % C4;
            float M = -INFINITY;
#pragma unroll
            for (int i = 0; i < NW; ++i) M = fmaxf(M, s_ml[buf][i][0][row]);
            float L = 0.f;
            float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int i = 0; i < NW; ++i) {
                const float wg = (M == -INFINITY) ? 0.f : exp2f(s_ml[buf][i][0][row] - M);
                L += wg * s_ml[buf][i][1][row];
                const float4 v = *reinterpret_cast<const float4*>(
                    reinterpret_cast<const float*>(smem + SM::OFF_XCHG + (size_t)(buf * NW + i) * SM::XCHG_WARP) + row * SM::OROW + c4 * 4);
                acc.x += wg * v.x; acc.y += wg * v.y; acc.z += wg * v.z; acc.w += wg * v.w;
            }
            if (n_parts == 1) {
                if (row < p.G) {
                    const float inv = L > 0.f ? 1.f / L : 0.f;
                    uint2 u;
                    u.x = pack_bf16(acc.x * inv, acc.y * inv);
                    u.y = pack_bf16(acc.z * inv, acc.w * inv);
                    *reinterpret_cast<uint2*>(obase + (size_t)row * D + c4 * 4) = u;
                }
            } else {
                __stcg(reinterpret_cast<float4*>(po + (size_t)row * D + c4 * 4), acc);
                if (c4 == 0) { __stcg(pml + row, M); __stcg(pml + 16 + row, L); }
            }
        }
    };
    // ---- row merge by the CTA that finished row r last: the row's n_parts partials (contiguous in the workspace) are
    // pulled into shared memory by bulk copies (TMA), mch at a time, and folded with a running (M, L, acc).  Landing area:
    // the idle K/V stages (16 partials per chunk) after the CTA's last segment, the second exchange buffer (4 per chunk)
    // for an earlier segment, whose successor's tiles are already in flight into the stages
    constexpr int MCH_STAGES = NW * SM::STAGE_BYTES / (16 * D * 4) > 16 ? 16 : NW * SM::STAGE_BYTES / (16 * D * 4);
    constexpr int MCH_XCHG = NW * SM::XCHG_WARP / (16 * D * 4);
    uint32_t phase_m = 0;
    auto row_merge = [&](int r, int n_parts, uint8_t* land_bytes, int mch) {
        float* land = reinterpret_cast<float*>(land_bytes);
        const int b = r / p.Hkv, g = r % p.Hkv;
        __nv_bfloat16* obase = p.O + (size_t)(b * p.Hq + g * p.G) * D;
        const float* rpo = p.part_O + (size_t)r * p.max_splits * 16 * D;
        const float* rml = p.part_ml + (size_t)r * p.max_splits * 32;
        constexpr int IPT = (16 * C4 + NT - 1) / NT;
        float LL[IPT];
        float4 acc[IPT];
#pragma unroll
        for (int j = 0; j < IPT; ++j) { LL[j] = 0.f; acc[j] = make_float4(0.f, 0.f, 0.f, 0.f); }
        if (tid < 16) s_run[tid] = -INFINITY;   // running row max
        __syncthreads();
        for (int i0 = 0; i0 < n_parts; i0 += mch) {
            const int n = min(mch, n_parts - i0);
            if (tid == 0) {
                fence_proxy_async_all();   // partials were written through the generic proxy (st.cg), read through the async proxy
                mbar_arrive_expect_tx(&bar_m, (uint32_t)n * (16 * D * 4 + 128));
                bulk_g2s(land, rpo + (size_t)i0 * 16 * D, (uint32_t)n * 16 * D * 4, &bar_m);
                bulk_g2s(s_pm, rml + (size_t)i0 * 32, (uint32_t)n * 128, &bar_m);
            }
            mbar_wait(&bar_m, phase_m);
            phase_m ^= 1;
            TRACE(7);
            // weights of the chunk, once per (partial, head row): s_w[i][row] = exp2(m_i - M_row), M_row the running max
            for (int e = tid; e < n * 16; e += NT) {
                const int row = e & 15;
                float mm = s_run[row];
                for (int i = 0; i < n; ++i) mm = fmaxf(mm, s_pm[i * 32 + row]);
                s_w[e] = (mm == -INFINITY) ? 0.f : exp2f(s_pm[(e >> 4) * 32 + row] - mm);
                if (e < 16) s_resc[row] = (mm == -INFINITY) ? 0.f : exp2f(s_run[row] - mm), s_newmax[row] = mm;
            }
            __syncthreads();
#pragma unroll
            for (int j = 0; j < IPT; ++j) {
                const int it = tid + j * NT;
                if (it >= 16 * C4) continue;
                const int row = it / C4, c4 = it % C4;
                const float resc = s_resc[row];
                LL[j] *= resc;
                acc[j].x *= resc; acc[j].y *= resc; acc[j].z *= resc; acc[j].w *= resc;
                const float* src = land + row * D + c4 * 4;
#pragma unroll 8
                for (int i = 0; i < n; ++i) {
                    const float wg = s_w[i * 16 + row];
                    LL[j] += wg * s_pm[i * 32 + 16 + row];
                    const float4 v = *reinterpret_cast<const float4*>(src + (size_t)i * 16 * D);
                    acc[j].x += wg * v.x; acc[j].y += wg * v.y; acc[j].z += wg * v.z; acc[j].w += wg * v.w;
                }
            }
            __syncthreads();
            if (tid < 16) s_run[tid] = s_newmax[tid];
            __syncthreads();   // the landing area may be overwritten by the next chunk
        }
#pragma unroll
        for (int j = 0; j < IPT; ++j) {
            const int it = tid + j * NT;
            if (it >= p.G * C4) continue;
            const int row = it / C4, c4 = it % C4;
            const float inv = LL[j] > 0.f ? 1.f / LL[j] : 0.f;
            uint2 u;
            u.x = pack_bf16(acc[j].x * inv, acc[j].y * inv);
            u.y = pack_bf16(acc[j].z * inv, acc[j].w * inv);
            *reinterpret_cast<uint2*>(obase + (size_t)row * D + c4 * 4) = u;
        }
    };
    // ---- publish this CTA's partial of row r and learn whether it finished the row last: CTA barrier, then one acq_rel
    // ticket at gpu scope (the release is cumulative over the CTA's st.cg partial writes ordered before it by the barrier;
    // the merging CTA acquires through the same atomic)
    auto publish = [&](int r, int n_parts) -> bool {
        __syncthreads();
        if (tid == 0) {
            unsigned int t;
            fence_proxy_async_all();
            asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(t) : "l"(p.tickets + r) : "memory");
            const bool last = t == (unsigned)n_parts - 1;
            if (last) p.tickets[r] = 0;   // re-arm
            s_last = last ? 1u : 0u;
        }
        __syncthreads();
        return s_last != 0;
    };
    int park_r = -1, park_part = 0, park_n = 1;

    int cur_r = -1, cur_s = 0;
    bool have = first_item(f_begin, cur_r, cur_s);
    if (lane == 0 && have) { issue_k(cur_r, cur_s); issue_v(cur_r, cur_s); }
    TRACE(1);

    for (int f = f_begin; f < f_end;) {
        const Seg sg = seg_at(f);
        const int r = sg.r;
        f += sg.s1 - sg.s0;
        const int first_cta = flat_owner(r * p.topk, p.quota, p.rem);
        const int n_parts = flat_owner((r + 1) * p.topk - 1, p.quota, p.rem) - first_cta + 1;
        const int part = blockIdx.x - first_cta;
        const int b = r / p.Hkv, g = r % p.Hkv;
        const int32_t* ids_row = p.ids + (size_t)r * p.topk;
        // tokens in row r's cache (varlen form): block j holds min(64, seq_row - 64 j) of them; INT_MAX = every block complete
        const int seq_row = VARLEN ? __ldg(p.seq_len + r) : 0x7fffffff;

        // Q fragments (A operand, 16 heads x D): rows gid and gid+8, zero beyond G
        uint32_t qa[KSTEPS][4];
        {
            const uint32_t* q0 = p.Q + ((size_t)(b * p.Hq + g * p.G + gid) * D) / 2;
            const uint32_t* q1 = q0 + (size_t)8 * D / 2;
            const bool v0 = gid < p.G, v1 = gid + 8 < p.G;
#pragma unroll
            for (int ks = 0; ks < KSTEPS; ++ks) {
                int c = ks * 8 + tig;  // uint32 index of columns ks*16 + tig*2
                qa[ks][0] = v0 ? __ldg(q0 + c) : 0u;
                qa[ks][1] = v1 ? __ldg(q1 + c) : 0u;
                qa[ks][2] = v0 ? __ldg(q0 + c + 4) : 0u;
                qa[ks][3] = v1 ? __ldg(q1 + c + 4) : 0u;
            }
        }

        float o[DT][4];
#pragma unroll
        for (int i = 0; i < DT; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
        float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
        bool first__ = true;
        (void)first__;

        while (have && cur_r == r) {   // this warp's items of the segment (a CTA's range meets a row in one segment only)
            // the item after this one: same segment, or the warp's first item of a later segment (staged across the merge)
            int nxt_r = r, nxt_s = cur_s + NW;
            bool have_n = true;
            if (nxt_s >= sg.s1) have_n = first_item(f, nxt_r, nxt_s);
            const int32_t id_cur = __ldg(ids_row + cur_s);
            const int n_tok = VARLEN ? min(S_BLK, seq_row - id_cur * S_BLK) : S_BLK;   // tokens of this block that exist (id <= 8191: no overflow)
            const bool valid = id_cur >= 0 && n_tok > 0;
            // ---- S = Q K^T
            mbar_wait(&bar_k[w], phase);
            if (first__) { TRACE(2); first__ = false; }
            float s[8][4];
            if (valid) {
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) {
                    s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.f;
                    const uint32_t row_addr = k_base + (nt * 8 + ri) * 128;
#pragma unroll
                    for (int kp = 0; kp < KSTEPS / 2; ++kp) {
                        const int c = kp * 4 + mi;  // 16-byte chunk of the D-row
                        uint32_t b0, b1, b2, b3;
                        ldmatrix_x4(row_addr + (c >> 3) * 8192 + (((c & 7) ^ ri) << 4), b0, b1, b2, b3);
                        mma_bf16_16816(s[nt], qa[2 * kp], b0, b1);
                        mma_bf16_16816(s[nt], qa[2 * kp + 1], b2, b3);
                    }
                }
            }
            if (VARLEN && valid && n_tok < S_BLK) {
                // the partly filled newest block: tokens >= n_tok do not exist.  Their scores are REPLACED (whatever bytes sit there,
                // NaN included) so that they get weight exp2(-inf) = 0.  Columns of s[nt][.]: tokens nt*8 + tig*2 + {0, 1}
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) {
                    const int c0 = nt * 8 + tig * 2;
                    if (c0 >= n_tok) s[nt][0] = s[nt][2] = -INFINITY;
                    if (c0 + 1 >= n_tok) s[nt][1] = s[nt][3] = -INFINITY;
                }
            }
            __syncwarp();
            if (lane == 0 && have_n) { fence_proxy_async_smem(); issue_k(nxt_r, nxt_s); }

            uint32_t pa[4][4];
            if (valid) {
                // ---- online softmax (exp2 domain), P rounded to bf16 feeds both the row sum and P V
                float mx0 = s[0][0], mx1 = s[0][2];
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) {
                    mx0 = fmaxf(mx0, fmaxf(s[nt][0], s[nt][1]));
                    mx1 = fmaxf(mx1, fmaxf(s[nt][2], s[nt][3]));
                }
                mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
                mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
                mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
                mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
                const float mn0 = fmaxf(m0, mx0 * p.scale_log2), mn1 = fmaxf(m1, mx1 * p.scale_log2);
                const float al0 = exp2f(m0 - mn0), al1 = exp2f(m1 - mn1);
                m0 = mn0; m1 = mn1;
                float rs0 = 0.f, rs1 = 0.f;
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) {
                    uint32_t u0 = pack_bf16(exp2f(fmaf(s[nt][0], p.scale_log2, -mn0)), exp2f(fmaf(s[nt][1], p.scale_log2, -mn0)));
                    uint32_t u1 = pack_bf16(exp2f(fmaf(s[nt][2], p.scale_log2, -mn1)), exp2f(fmaf(s[nt][3], p.scale_log2, -mn1)));
                    rs0 += bf16_lo(u0) + bf16_hi(u0);
                    rs1 += bf16_lo(u1) + bf16_hi(u1);
                    pa[nt >> 1][(nt & 1) * 2 + 0] = u0;
                    pa[nt >> 1][(nt & 1) * 2 + 1] = u1;
                }
                l0 = l0 * al0 + rs0;
                l1 = l1 * al1 + rs1;
#pragma unroll
                for (int i = 0; i < DT; ++i) { o[i][0] *= al0; o[i][1] *= al0; o[i][2] *= al1; o[i][3] *= al1; }
            }

            // ---- O += P V
            mbar_wait(&bar_v[w], phase);
            if (VARLEN && valid && n_tok < S_BLK) {
                // weight 0 times a NaN / Inf left behind the tail would still poison O: zero the V rows that do not exist in the
                // warp's stage (a row is 128 contiguous bytes per 64-column box whatever the swizzle); generic-proxy stores, ordered
                // before the next TMA write into the stage by the fence in front of issue_v
                const int n_chunks = (S_BLK - n_tok) * HALVES * 8;   // 16-byte chunks
                for (int c = lane; c < n_chunks; c += 32) {
                    const int row = n_tok + c / (HALVES * 8), h = (c / 8) % HALVES, q16 = c % 8;
                    *reinterpret_cast<int4*>(stage + SM::TILE_BYTES + h * 8192 + row * 128 + q16 * 16) = make_int4(0, 0, 0, 0);
                }
                __syncwarp();
            }
            if (valid) {
#pragma unroll
                for (int kt = 0; kt < 4; ++kt) {
                    const uint32_t row_addr = v_base + (kt * 16 + (mi & 1) * 8 + ri) * 128;
#pragma unroll
                    for (int dp = 0; dp < DT / 2; ++dp) {
                        const int c = dp * 2 + (mi >> 1);
                        uint32_t b0, b1, b2, b3;
                        ldmatrix_x4_trans(row_addr + (c >> 3) * 8192 + (((c & 7) ^ ri) << 4), b0, b1, b2, b3);
                        mma_bf16_16816(o[2 * dp], pa[kt], b0, b1);
                        mma_bf16_16816(o[2 * dp + 1], pa[kt], b2, b3);
                    }
                }
            }
            __syncwarp();
            if (lane == 0 && have_n) { fence_proxy_async_smem(); issue_v(nxt_r, nxt_s); }
            phase ^= 1;
            cur_r = nxt_r;
            cur_s = nxt_s;
            have = have_n;
        }
        TRACE(3);
        // ---- warp partial -> exchange buffer 0
        l0 += __shfl_xor_sync(0xffffffffu, l0, 1);
        l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
        l1 += __shfl_xor_sync(0xffffffffu, l1, 1);
        l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
        float* wo = reinterpret_cast<float*>(smem + SM::OFF_XCHG + (size_t)w * SM::XCHG_WARP);
#pragma unroll
        for (int i = 0; i < DT; ++i) {
            *reinterpret_cast<float2*>(wo + gid * SM::OROW + i * 8 + tig * 2) = make_float2(o[i][0], o[i][1]);
            *reinterpret_cast<float2*>(wo + (gid + 8) * SM::OROW + i * 8 + tig * 2) = make_float2(o[i][2], o[i][3]);
        }
        if (tig == 0) {
            s_ml[0][w][0][gid] = m0; s_ml[0][w][1][gid] = l0;
            s_ml[0][w][0][gid + 8] = m1; s_ml[0][w][1][gid + 8] = l1;
        }
        if (f >= f_end && n_parts > 1) {   // the CTA's last segment: finished below, when the stages are idle
            park_r = r; park_part = part; park_n = n_parts;
            break;
        }
        __syncthreads();
        cta_merge(0, r, part, n_parts);
        if (n_parts > 1 && publish(r, n_parts))
            row_merge(r, n_parts, smem + SM::OFF_XCHG + (size_t)NW * SM::XCHG_WARP, MCH_XCHG);
        __syncthreads();   // exchange buffer 0 is free again
    }
    if (park_r < 0) return;
    __syncthreads();
    TRACE(3);
    if (CL) {
        // ---- cluster reduction of the row's n = park_n partials.  Landing area (exchange buffer 1, unused in this mode):
        // land[p][lrow][D] fp32 and ml[p][lrow][2], p = source CTA, lrow = head row within this CTA's 16 / n rows.
        const int n = park_n, part = park_part, r = park_r;
        const int rows_per = 16 / n;
        float* land = reinterpret_cast<float*>(smem + SM::OFF_XCHG + (size_t)NW * SM::XCHG_WARP);
        float* land_ml = land + 16 * D;
        const uint32_t land_u32 = smem_u32(land), ml_u32 = smem_u32(land_ml), red_u32 = smem_u32(&bar_red);
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");   // pairs with the arrive at kernel start
        for (int it = tid; it < 16 * C4; it += NT) {
            const int row = it / C4, c4 = it % C4;
            float M = -INFINITY;
#pragma unroll
            for (int i = 0; i < NW; ++i) M = fmaxf(M, s_ml[0][i][0][row]);
            float L = 0.f;
            float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int i = 0; i < NW; ++i) {
                const float wg = (M == -INFINITY) ? 0.f : exp2f(s_ml[0][i][0][row] - M);
                L += wg * s_ml[0][i][1][row];
                const float4 v = *reinterpret_cast<const float4*>(
                    reinterpret_cast<const float*>(smem + SM::OFF_XCHG + (size_t)i * SM::XCHG_WARP) + row * SM::OROW + c4 * 4);
                acc.x += wg * v.x; acc.y += wg * v.y; acc.z += wg * v.z; acc.w += wg * v.w;
            }
            // asynchronous stores into the owner's landing area that count their bytes on the owner's barrier: no release
            // fence and no closing cluster barrier -- the owner waits for "16 x (D x 4 + 8) bytes have landed"
            const uint32_t owner = (uint32_t)(row / rows_per), lrow = (uint32_t)(row % rows_per);
            uint32_t dst, dml, dbar;
            asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(dbar) : "r"(red_u32), "r"(owner));
            asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(dst) : "r"(land_u32 + ((part * rows_per + lrow) * D + c4 * 4) * 4), "r"(owner));
            asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1, %2, %3, %4}, [%5];" ::"r"(dst), "f"(acc.x),
                         "f"(acc.y), "f"(acc.z), "f"(acc.w), "r"(dbar)
                         : "memory");
            if (c4 == 0) {
                asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(dml) : "r"(ml_u32 + ((part * rows_per + lrow) * 2) * 4), "r"(owner));
                asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f32 [%0], {%1, %2}, [%3];" ::"r"(dml), "f"(M), "f"(L), "r"(dbar)
                             : "memory");
            }
        }
        TRACE(4);
        mbar_wait(&bar_red, 0);
        TRACE(5);
        const int b = r / p.Hkv, g = r % p.Hkv;
        __nv_bfloat16* obase = p.O + (size_t)(b * p.Hq + g * p.G) * D;
        for (int it = tid; it < rows_per * C4; it += NT) {
            const int lrow = it / C4, c4 = it % C4;
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
        TRACE(6);
        return;
    }
    cta_merge(0, park_r, park_part, park_n);
    TRACE(4);
    const bool owes_merge = publish(park_r, park_n);
    TRACE(5);
    if (owes_merge) row_merge(park_r, park_n, smem, MCH_STAGES);
    TRACE(6);
}

// Launch shape: 4 consumer warps (= 4 x 32 KiB K/V stages at D = 128), one CTA per SM (128 KiB of tiles in flight per SM).
constexpr int ATT_NW = 4;

template <int D, bool CL, bool VL = false>
int launch(sparda_ctx* ctx, const CUtensorMap* map, const AttnParams& p, int C, int cluster, cudaStream_t st) {
    auto kern = sparse_decode_kernel<D, ATT_NW, 1, CL, VL>;
    constexpr int smem = AttnSmem<D, ATT_NW>::TOTAL;
    sparda_kernel_state& ks = ctx->kstate[(VL ? (CL ? SPARDA_K_ATTN_VL_CL_128 : SPARDA_K_ATTN_VL_128) : (CL ? SPARDA_K_ATTN_CL_128 : SPARDA_K_ATTN_128)) +
                                          (D == 128 ? 0 : 1)];
    if (!ks.attr_set) {
        SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        if (CL) SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));   // clusters of 16
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
    lc.blockDim = dim3(ATT_NW * 32, 1, 1);
    lc.dynamicSmemBytes = smem;
    lc.stream = st;
    if (CL) {
        // a cluster needs `cluster` SMs of one GPC at the same time (one CTA per SM): use this path only when every row's
        // cluster is resident in one wave, else the second wave costs more than the reduction saves (batch 8, 16 x 8 CTAs)
        if (ks.max_clusters[cluster] == 0) {   // asked once per context and cluster size (the shared-memory size is fixed)
            int n = 0;
            if (cudaOccupancyMaxActiveClusters(&n, kern, &lc) != cudaSuccess) n = -1;
            (void)cudaGetLastError();
            ks.max_clusters[cluster] = n > 0 ? n : -1;
        }
        if (ks.max_clusters[cluster] * cluster < C) return 1;   // caller falls back to the workspace reduction
    }
    lc.numAttrs = sparda_use_pdl(ctx) ? 2 : 1;
    SPARDA_CUDA_TRY(ctx, cudaLaunchKernelEx(&lc, kern, *map, p));
    return SPARDA_OK;
}

}  // namespace

// Grid size of the flat split.  attn_splits = s > 0: s CTAs per row.  attn_splits = 0 (measured on B200, 128K shapes,
// batch 4..32): a row-aligned split wins whenever one exists -- s CTAs per row with s a divisor of topk, s <= 8 (few
// partials per row keep the row merge short) and s*R <= SM count, the largest such grid (batch 32: 2 x 64 = 128 CTAs,
// 0.73 of the HBM peak against 0.64 for 148 row-spanning CTAs).  Otherwise (R > SM count, or topk without a useful
// divisor) one CTA per SM over the flat list, at least one slot per consumer warp.  Always <= W and within the workspace.
int sparda_resolve_attn_ctas(const sparda_ctx* ctx, int topk) {
    const long long W = (long long)ctx->R * topk;
    long long C;
    if (ctx->cfg.attn_splits > 0) {
        C = (long long)ctx->cfg.attn_splits * ctx->R;
    } else {
        long long flat = ctx->sm_count;
        if (flat > 8LL * ctx->R) flat = 8LL * ctx->R;
        const long long cap = (W + ATT_NW - 1) / ATT_NW;
        if (flat > cap) flat = cap;
        long long aligned = 0;
        for (int s = 1; s <= 8 && s <= topk; ++s)
            if (topk % s == 0 && (long long)s * ctx->R <= ctx->sm_count) aligned = (long long)s * ctx->R;
        // up to 4 rows (batch 1-2): clusters of 16 (non-portable size), topk / 16 slots per CTA -- at k = 64 every tile of the
        // launch is in flight at once, one DRAM round trip per warp (measured, 128K shapes: batch 2 7.2 -> 6.5 us, batch 1
        // 7.1 -> 5.9 us).  From 8 rows on the device cannot keep all clusters of 16 resident (one 200 KB CTA per SM).
        if (topk % 16 == 0 && ctx->R <= 4) aligned = 16LL * ctx->R;
        C = (aligned * 5 >= flat * 3) ? aligned : flat;
    }
    // workspace: a row meets at most ceil(topk / quota) + 1 CTAs, quota = floor(W / C); keep that <= max_splits
    const long long quota_min = (topk + ctx->max_splits - 2) / (ctx->max_splits - 1);
    if (C > W / quota_min) C = W / quota_min;
    if (C > W) C = W;
    if (C < 1) C = 1;
    return (int)C;
}

int sparda_resolve_splits(const sparda_ctx* ctx, int topk) {
    return (sparda_resolve_attn_ctas(ctx, topk) + ctx->R - 1) / ctx->R;
}

int sparda_launch_attn(sparda_ctx* ctx, const void* Q, const void* pool, const int32_t* ids, const int32_t* seq_len, int topk, int indexed,
                       int n_slots, void* O, cudaStream_t st) {
    if (ctx->cfg.attn_impl == 1 && !seq_len) {   // the tcgen05 (swap-AB) experiment; shapes outside its range (and the varlen form) fall through
        const int rc5 = sparda_launch_attn_tc5(ctx, Q, pool, ids, topk, indexed, n_slots, O, st);
        if (rc5 != 1) return rc5;
    }
    const int D = ctx->cfg.head_dim;
    const uint64_t rows = (uint64_t)ctx->R * n_slots * 2 * S_BLK;
    CUtensorMap map;
    int rc = sparda_get_tmap(ctx, pool, rows, D, S_BLK, &map);
    if (rc) return rc;
    AttnParams p;
    p.Q = (const uint32_t*)Q;
    p.ids = ids;
    p.seq_len = seq_len;
    p.O = (__nv_bfloat16*)O;
    p.part_O = ctx->part_O;
    p.part_ml = ctx->part_ml;
    p.tickets = ctx->tickets;
    p.topk = topk;
    p.indexed = indexed;
    p.n_slots = n_slots;
    p.Hq = ctx->cfg.n_q_heads;
    p.Hkv = ctx->cfg.n_kv_heads;
    p.G = ctx->G;
    p.max_splits = ctx->max_splits;
    p.W = ctx->R * topk;
    p.scale_log2 = 1.4426950408889634f / sqrtf((float)D);
    const int C = sparda_resolve_attn_ctas(ctx, topk);
    p.quota = p.W / C;
    p.rem = p.W % C;
    // row-aligned split with 2, 4, 8 or 16 CTAs per row: reduce the partials inside a cluster (distributed shared memory)
    const int s_per = p.quota > 0 && p.rem == 0 && topk % p.quota == 0 ? topk / p.quota : 0;
    const bool cl = (s_per == 2 || s_per == 4 || s_per == 8 || s_per == 16) && (long long)s_per * ctx->R == C;
    rc = 1;
    int used_cl = 0;
    if (cl) {
        // When the device cannot keep all R clusters of s_per CTAs resident (batch 8: 16 clusters of 8 with one 200 KB CTA per
        // SM), half as many CTAs per row in clusters that do fit beat the same CTA count reduced through the L2 workspace
        // (measured, batch 8: 128 CTAs + ticket 11.9 us; 64 CTAs in clusters of 4: see DESIGN.md 5.3).  The automatic split
        // only: an explicit cfg.attn_splits is honoured as given.
        for (int s = s_per; s >= 2 && rc == 1; s /= 2) {
            if (topk % s != 0) break;
            AttnParams q = p;
            const int Cs = s * ctx->R;
            q.quota = q.W / Cs;
            q.rem = 0;
            if (seq_len) rc = D == 128 ? launch<128, true, true>(ctx, &map, q, Cs, s, st) : launch<64, true, true>(ctx, &map, q, Cs, s, st);
            else rc = D == 128 ? launch<128, true>(ctx, &map, q, Cs, s, st) : launch<64, true>(ctx, &map, q, Cs, s, st);
            if (rc != 1) used_cl = s;
            if (ctx->cfg.attn_splits > 0) break;
        }
    }
    if (rc == 1 && seq_len) rc = D == 128 ? launch<128, false, true>(ctx, &map, p, C, 1, st) : launch<64, false, true>(ctx, &map, p, C, 1, st);
    else if (rc == 1) rc = D == 128 ? launch<128, false>(ctx, &map, p, C, 1, st) : launch<64, false>(ctx, &map, p, C, 1, st);
    if (rc) return rc;
    SPARDA_CUDA_TRY(ctx, cudaGetLastError());
    ctx->last_attn_cluster = used_cl;
    ctx->launches++;
    return SPARDA_OK;
}

// =================================================================================================================
// sparda_sparse_decode_noalloc (include/sparda.h): the attention above for callers that may not allocate device
// memory -- an engine that gave all of HBM to its own pool, a decode loop that cannot take cudaMalloc's device-wide
// synchronisation, a plug-in with no set-up hook.  Such a caller cannot use sparda_create (cudaMalloc, stream and event
// creation), so this entry point takes no context: the launcher state a context would hold sits in a host-side table with
// one entry per device, and the split-K workspace (CTA partials + per-row tickets) is the fixed array below instead of
// cudaMalloc'ed memory.  The kernel is sparse_decode_kernel<D, 4, 1, false, false> unchanged -- the flat split whose row
// partials are merged by the last CTA to finish the row -- with its three workspace pointers aimed into the array.
//
// The array is part of this translation unit's device image: the driver places it on every GPU that loads the image and
// keeps it until the process exits.  In HOST code the name `g_noalloc_scratch` is only a handle for the runtime's symbol
// table -- it is not a device address, and a kernel given `&g_noalloc_scratch[0]` from the host would fault or scribble
// over host memory.  The device address is asked for once per device with cudaGetSymbolAddress (noalloc_setup) and that
// pointer is what the kernel receives.
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>

static __device__ __align__(256) unsigned char g_noalloc_scratch[SPARDA_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int NA_MAX_DEVICES = 16;   // device ordinals this table covers
constexpr size_t NA_PART_O_BYTES = (size_t)SPARDA_NOALLOC_MAX_PARTIALS * 16 * 128 * sizeof(float);   // [partials][16][D <= 128]
constexpr size_t NA_PART_ML_BYTES = (size_t)SPARDA_NOALLOC_MAX_PARTIALS * 2 * 16 * sizeof(float);    // [partials][2][16]
constexpr size_t NA_TICKET_BYTES = (size_t)SPARDA_NOALLOC_MAX_ROWS * sizeof(unsigned int);           // [rows]
static_assert(NA_PART_O_BYTES + NA_PART_ML_BYTES + NA_TICKET_BYTES == SPARDA_NOALLOC_SCRATCH_BYTES,
              "sparda.h states the array's size; keep the layout and the figure together");
static_assert(SPARDA_NOALLOC_MAX_PARTIALS >= 2 * SPARDA_NOALLOC_MAX_ROWS,
              "a row of the flat split may meet two CTAs: every admitted R needs at least two partial slots per row");

struct NoallocDevice {
    bool ready;
    unsigned char* scratch;   // DEVICE address of g_noalloc_scratch on this device (cudaGetSymbolAddress)
    sparda_ctx ctx;           // launcher state only (descriptor cache, attribute flags, shape of the current call): no device memory
};
NoallocDevice g_na[NA_MAX_DEVICES];   // host memory, static: nothing is allocated on the host either
std::mutex g_na_lock;
thread_local char g_na_err[384];

int na_fail(int code, const char* fmt, ...) __attribute__((format(printf, 2, 3)));
int na_fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_na_err, sizeof(g_na_err), fmt, ap);
    va_end(ap);
    return code;
}
int na_fail_cuda(cudaError_t e, const char* where) {
    (void)cudaGetLastError();
    return na_fail(SPARDA_ECUDA, "%s: %s (%s)", cudaGetErrorName(e), cudaGetErrorString(e), where);
}

// Once per device, with that device current.  Everything here is a query or a per-function attribute: no cudaMalloc, no
// stream, no event.  Run it (= make the first call on the device) before any stream capture begins.
int noalloc_setup(NoallocDevice& d, int dev) {
    int major = 0, sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return na_fail_cuda(e, "cudaDeviceGetAttribute");
    if (major != 10) return na_fail(SPARDA_EUNSUPPORTED, "device %d has compute capability %d.x; libsparda's kernels are sm_100a only", dev, major);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess) return na_fail_cuda(e, "cudaGetDriverEntryPoint(cuTensorMapEncodeTiled)");
    if (qres != cudaDriverEntryPointSuccess || !fn) return na_fail(SPARDA_EUNSUPPORTED, "the driver does not export cuTensorMapEncodeTiled");
    unsigned char* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch);   // the array's address ON THIS DEVICE
    if (e != cudaSuccess) return na_fail_cuda(e, "cudaGetSymbolAddress(g_noalloc_scratch)");
    if (!ptr) return na_fail(SPARDA_ECUDA, "cudaGetSymbolAddress(g_noalloc_scratch) returned a null device address");
    e = cudaFuncSetAttribute(sparse_decode_kernel<128, ATT_NW, 1, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, AttnSmem<128, ATT_NW>::TOTAL);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(sparse_decode_kernel<64, ATT_NW, 1, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, AttnSmem<64, ATT_NW>::TOTAL);
    if (e != cudaSuccess) return na_fail_cuda(e, "cudaFuncSetAttribute(sparse_decode_kernel, MaxDynamicSharedMemorySize)");
    memset(&d.ctx, 0, sizeof(d.ctx));
    d.ctx.device = dev;
    d.ctx.sm_count = sms;
    d.ctx.encode_fn = fn;
    d.ctx.cfg.block_size = S_BLK;
    d.ctx.cfg.no_pdl = 1;   // plain stream order behind the ticket memset
    d.ctx.kstate[SPARDA_K_ATTN_128].attr_set = true;
    d.ctx.kstate[SPARDA_K_ATTN_64].attr_set = true;
    d.scratch = ptr;
    d.ready = true;
    return SPARDA_OK;
}

}  // namespace

extern "C" const char* sparda_noalloc_last_error(void) { return g_na_err; }

extern "C" int sparda_sparse_decode_noalloc(int batch, int n_q_heads, int n_kv_heads, int head_dim, const void* Q, const void* dev_pool,
                                            const int32_t* ids, int topk, int pool_is_indexed, int n_slots, void* O, void* stream) {
    g_na_err[0] = 0;
    // ---- shape and pointer checks: no CUDA call before they pass
    if (!sparda_aligned(Q, 16) || !sparda_aligned(dev_pool, 16) || !sparda_aligned(O, 16) || !sparda_aligned(ids, 4))
        return na_fail(SPARDA_EINVAL, "null or misaligned pointer (Q, dev_pool, O: 16 bytes; ids: 4 bytes)");
    if (batch < 1 || n_kv_heads < 1 || n_q_heads < 1 || n_q_heads % n_kv_heads != 0)
        return na_fail(SPARDA_EINVAL, "batch %d, n_q_heads %d, n_kv_heads %d: need positive counts and n_q_heads a multiple of n_kv_heads", batch, n_q_heads, n_kv_heads);
    const int G = n_q_heads / n_kv_heads;
    if (!(G == 1 || G == 2 || G == 4 || G == 8 || G == 16)) return na_fail(SPARDA_EINVAL, "G = n_q_heads / n_kv_heads = %d: supported 1, 2, 4, 8, 16", G);
    if (head_dim != 64 && head_dim != 128) return na_fail(SPARDA_EINVAL, "head_dim %d: supported 64 and 128", head_dim);
    if (topk < 1 || topk > 256) return na_fail(SPARDA_EINVAL, "topk %d: supported 1..256", topk);
    if (pool_is_indexed ? (n_slots < 1 || n_slots > 8192) : (n_slots != topk))
        return na_fail(SPARDA_EINVAL, "n_slots %d: 1..8192 blocks per row for an indexed cache, else exactly topk (%d)", n_slots, topk);
    const long long R = (long long)batch * n_kv_heads;
    if (R > SPARDA_NOALLOC_MAX_ROWS)
        return na_fail(SPARDA_ELIMIT,
                       "batch * n_kv_heads = %lld rows, but the built-in scratch array holds tickets and split-K partials for at most "
                       "SPARDA_NOALLOC_MAX_ROWS = %d rows (%d bytes in all): split the batch over several calls on one stream, or use "
                       "sparda_create + sparda_sparse_decode where allocating is allowed",
                       R, SPARDA_NOALLOC_MAX_ROWS, (int)SPARDA_NOALLOC_SCRATCH_BYTES);

    std::lock_guard<std::mutex> guard(g_na_lock);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail_cuda(e, "cudaGetDevice");
    if (dev < 0 || dev >= NA_MAX_DEVICES) return na_fail(SPARDA_ELIMIT, "device ordinal %d: the per-device table covers ordinals 0..%d", dev, NA_MAX_DEVICES - 1);
    NoallocDevice& d = g_na[dev];
    if (!d.ready) {
        const int rc = noalloc_setup(d, dev);
        if (rc) return rc;
    }

    // ---- the shape a context would carry, for this call
    sparda_ctx* ctx = &d.ctx;
    ctx->cfg.batch = batch;
    ctx->cfg.n_q_heads = n_q_heads;
    ctx->cfg.n_kv_heads = n_kv_heads;
    ctx->cfg.head_dim = head_dim;
    ctx->cfg.topk = topk;
    ctx->R = (int)R;
    ctx->G = G;
    {   // partial slots per row: what sparda_create would give (ceil(2 * SMs / R) CTAs per row + 2), cut to the array's capacity;
        // sparda_resolve_attn_ctas then keeps every row within that many CTAs (>= 2 for every admitted R)
        int per_row = (2 * ctx->sm_count + ctx->R - 1) / ctx->R;
        if (per_row > topk) per_row = topk;
        ctx->max_splits = per_row + 2;
        if (ctx->max_splits > SPARDA_NOALLOC_MAX_PARTIALS / ctx->R) ctx->max_splits = SPARDA_NOALLOC_MAX_PARTIALS / ctx->R;
    }
    ctx->part_O = reinterpret_cast<float*>(d.scratch);
    ctx->part_ml = reinterpret_cast<float*>(d.scratch + NA_PART_O_BYTES);
    ctx->tickets = reinterpret_cast<unsigned int*>(d.scratch + NA_PART_O_BYTES + NA_PART_ML_BYTES);

    cudaStream_t st = (cudaStream_t)stream;
    CUtensorMap map;
    if (sparda_get_tmap(ctx, dev_pool, (uint64_t)ctx->R * n_slots * 2 * S_BLK, head_dim, S_BLK, &map) != SPARDA_OK)
        return na_fail(SPARDA_ECUDA, "%s", ctx->cuda_err);
    AttnParams p;
    p.Q = (const uint32_t*)Q;
    p.ids = ids;
    p.seq_len = nullptr;
    p.O = (__nv_bfloat16*)O;
    p.part_O = ctx->part_O;
    p.part_ml = ctx->part_ml;
    p.tickets = ctx->tickets;
    p.topk = topk;
    p.indexed = pool_is_indexed ? 1 : 0;
    p.n_slots = n_slots;
    p.Hq = n_q_heads;
    p.Hkv = n_kv_heads;
    p.G = G;
    p.max_splits = ctx->max_splits;
    p.W = ctx->R * topk;
    p.scale_log2 = 1.4426950408889634f / sqrtf((float)head_dim);
    const int C = sparda_resolve_attn_ctas(ctx, topk);
    p.quota = p.W / C;
    p.rem = p.W % C;
    // The array keeps the previous call's contents.  Partials are written before they are read within one launch, so they need
    // no clearing; the tickets count arrivals from zero, and a launch that was cut short (or a foreign write) must not leak
    // into this one: clear this call's R tickets in stream order in front of the kernel.
    e = cudaMemsetAsync(ctx->tickets, 0, (size_t)ctx->R * sizeof(unsigned int), st);
    if (e != cudaSuccess) return na_fail_cuda(e, "cudaMemsetAsync(tickets)");
    const int rc = head_dim == 128 ? launch<128, false>(ctx, &map, p, C, 1, st) : launch<64, false>(ctx, &map, p, C, 1, st);
    if (rc) return na_fail(rc, "%s", ctx->cuda_err);
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail_cuda(e, "sparse_decode_kernel launch");
    ctx->launches++;
    return SPARDA_OK;
}
