// Block-sparse GQA decode attention over the gathered blocks (a5) and over a device-resident cache
// addressed by block id (a6, layer 0).  Eq.5, Alg.2 l.7:
//   O_h = softmax_t( q_h . k_t / sqrt(D) ) V   over every token t of every selected block of row r = b*Hkv + h/G.
//
// Split-K flash-decode.  Grid (splits, R); a CTA owns a contiguous range of pool slots of one row and has
// SPARDA_ATTN_WARPS consumer warps, each with its own shared-memory stage (one block's K and V tiles,
// 2*S*D*2 bytes).  Lane 0 of a warp stages the warp's next block with TMA tensor-map loads
// (cp.async.bulk.tensor.2d, 64x64 boxes, 128-byte swizzle so ldmatrix is bank-conflict free) completing
// on per-stage mbarriers (K and V separately: QK^T starts when K lands, and the next K load is issued
// as soon as QK^T has consumed the tile).  The group's G <= 16 query heads are the M = 16 rows of
// mma.sync.m16n8k16 (bf16 in, fp32 accumulate): S = Q K^T (16 x 64 per block), online softmax in the
// exp2 domain, O += P V.  Warp partials (m, l, O) are merged through shared memory, CTA partials through
// an L2-resident workspace by the last CTA of the row (ticket), which rounds once to bf16.
// HBM-bound by design: 16 FLOP per KV byte at G = 16; the tensor pipe idles most of the time.
#include "sparda_internal.cuh"

namespace {

using namespace sparda;

constexpr int NW = SPARDA_ATTN_WARPS;
constexpr int ATT_THREADS = NW * 32;
constexpr int S_BLK = 64;

template <int D>
struct AttnSmem {
    static constexpr int TILE_BYTES = S_BLK * D * 2;        // one K (or V) tile
    static constexpr int STAGE_BYTES = 2 * TILE_BYTES;      // K then V
    static constexpr int OROW = D + 4;                      // padded fp32 row of the warp partial
    static constexpr int TOTAL = NW * STAGE_BYTES + 1024;   // + slack for 1024-byte alignment
    static_assert(16 * OROW * 4 <= STAGE_BYTES, "warp partial must fit in the warp's own stage");
};

struct AttnParams {
    const uint32_t* Q;     // bf16 pairs
    const int32_t* ids;
    __nv_bfloat16* O;
    float* part_O;
    float* part_ml;
    unsigned int* tickets;
    int topk, indexed, n_slots, Hq, Hkv, G, splits, max_splits;
    float scale_log2;
};

// merge n partials {m[i], l[i], o[i]} -> (M, L, acc); weights exp2(m_i - M)
template <int D>
__global__ void __launch_bounds__(ATT_THREADS, 1) sparse_decode_kernel(const __grid_constant__ CUtensorMap tmap, AttnParams p) {
    using SM = AttnSmem<D>;
    constexpr int KSTEPS = D / 16;  // k-steps of Q K^T
    constexpr int DT = D / 8;       // n-tiles of P V
    constexpr int HALVES = D / 64;  // 64-element TMA boxes per row
    extern __shared__ uint8_t smem_raw[];
    __shared__ uint64_t bar_k[NW], bar_v[NW];
    __shared__ float s_ml[NW][2][16];
    __shared__ unsigned int s_ticket;

    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int r = blockIdx.y, split = blockIdx.x;
    const int b = r / p.Hkv, g = r % p.Hkv;
    const int gid = lane >> 2, tig = lane & 3;

    if (tid == 0) {
        for (int i = 0; i < NW; ++i) { mbar_init(&bar_k[i], 1); mbar_init(&bar_v[i], 1); }
        mbar_fence_init();
        fence_proxy_async_smem();
        tma_prefetch_desc(&tmap);
    }
    __syncthreads();

    const int bps = (p.topk + p.splits - 1) / p.splits;
    const int slot_begin = split * bps;
    const int slot_end = min(p.topk, slot_begin + bps);
    const int32_t* ids_row = p.ids + (size_t)r * p.topk;

    uint8_t* stage = smem + (size_t)w * SM::STAGE_BYTES;
    const uint32_t k_base = smem_u32(stage), v_base = k_base + SM::TILE_BYTES;

    auto next_valid = [&](int s) {
        while (s < slot_end && __ldg(ids_row + s) < 0) s += NW;
        return s;
    };
    auto tile_row = [&](int slot, int plane) -> int {
        int idx = p.indexed ? __ldg(ids_row + slot) : slot;
        return (((r * p.n_slots + idx) * 2 + plane) * S_BLK);
    };
    auto issue_k = [&](int slot) {
        mbar_arrive_expect_tx(&bar_k[w], SM::TILE_BYTES);
#pragma unroll
        for (int h = 0; h < HALVES; ++h) tma_load_2d(stage + h * 8192, &tmap, h * 64, tile_row(slot, 0), &bar_k[w]);
    };
    auto issue_v = [&](int slot) {
        mbar_arrive_expect_tx(&bar_v[w], SM::TILE_BYTES);
#pragma unroll
        for (int h = 0; h < HALVES; ++h)
            tma_load_2d(stage + SM::TILE_BYTES + h * 8192, &tmap, h * 64, tile_row(slot, 1), &bar_v[w]);
    };

    int cur = next_valid(slot_begin + w);
    if (lane == 0 && cur < slot_end) { issue_k(cur); issue_v(cur); }

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
    uint32_t phase = 0;

    // per-lane ldmatrix row offsets (swizzle: 16-byte chunk index ^= row & 7; rows are 128 B inside a box)
    const int mi = lane >> 3, ri = lane & 7;

    while (cur < slot_end) {
        const int nxt = next_valid(cur + NW);
        // ---- S = Q K^T
        mbar_wait(&bar_k[w], phase);
        float s[8][4];
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
        __syncwarp();
        if (lane == 0 && nxt < slot_end) { fence_proxy_async_smem(); issue_k(nxt); }

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
        uint32_t pa[4][4];
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

        // ---- O += P V
        mbar_wait(&bar_v[w], phase);
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
        __syncwarp();
        if (lane == 0 && nxt < slot_end) { fence_proxy_async_smem(); issue_v(nxt); }
        phase ^= 1;
        cur = nxt;
    }

    // ---- warp partial -> this warp's own (now idle) stage
    l0 += __shfl_xor_sync(0xffffffffu, l0, 1);
    l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
    l1 += __shfl_xor_sync(0xffffffffu, l1, 1);
    l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
    float* wo = reinterpret_cast<float*>(stage);
#pragma unroll
    for (int i = 0; i < DT; ++i) {
        *reinterpret_cast<float2*>(wo + gid * SM::OROW + i * 8 + tig * 2) = make_float2(o[i][0], o[i][1]);
        *reinterpret_cast<float2*>(wo + (gid + 8) * SM::OROW + i * 8 + tig * 2) = make_float2(o[i][2], o[i][3]);
    }
    if (tig == 0) {
        s_ml[w][0][gid] = m0; s_ml[w][1][gid] = l0;
        s_ml[w][0][gid + 8] = m1; s_ml[w][1][gid + 8] = l1;
    }
    __syncthreads();

    // ---- CTA merge: thread -> (row, 4-column groups); 8 threads per row
    const int row = tid >> 3, cg = tid & 7;
    constexpr int NCG = D / 32;  // float4 groups per thread
    float M = -INFINITY;
#pragma unroll
    for (int i = 0; i < NW; ++i) M = fmaxf(M, s_ml[i][0][row]);
    float wgt[NW], L = 0.f;
#pragma unroll
    for (int i = 0; i < NW; ++i) {
        wgt[i] = (M == -INFINITY) ? 0.f : exp2f(s_ml[i][0][row] - M);
        L += wgt[i] * s_ml[i][1][row];
    }
    float4 acc[NCG];
#pragma unroll
    for (int j = 0; j < NCG; ++j) {
        acc[j] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int i = 0; i < NW; ++i) {
            const float4 v = *reinterpret_cast<const float4*>(reinterpret_cast<const float*>(smem + (size_t)i * SM::STAGE_BYTES) +
                                                               row * SM::OROW + cg * 4 + j * 32);
            acc[j].x += wgt[i] * v.x; acc[j].y += wgt[i] * v.y; acc[j].z += wgt[i] * v.z; acc[j].w += wgt[i] * v.w;
        }
    }
    __nv_bfloat16* orow = p.O + (size_t)(b * p.Hq + g * p.G + row) * D;
    auto store_out = [&](const float4 (&a)[NCG], float Lsum) {
        const float inv = Lsum > 0.f ? 1.f / Lsum : 0.f;
#pragma unroll
        for (int j = 0; j < NCG; ++j) {
            uint2 u;
            u.x = pack_bf16(a[j].x * inv, a[j].y * inv);
            u.y = pack_bf16(a[j].z * inv, a[j].w * inv);
            *reinterpret_cast<uint2*>(orow + cg * 4 + j * 32) = u;
        }
    };
    if (p.splits == 1) {
        if (row < p.G) store_out(acc, L);
        return;
    }
    if (row < p.G) {
        float* po = p.part_O + ((size_t)(r * p.max_splits + split) * 16 + row) * D;
#pragma unroll
        for (int j = 0; j < NCG; ++j) __stcg(reinterpret_cast<float4*>(po + cg * 4 + j * 32), acc[j]);
        if (cg == 0) {
            float* pml = p.part_ml + (size_t)(r * p.max_splits + split) * 32;
            __stcg(pml + row, M);
            __stcg(pml + 16 + row, L);
        }
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) s_ticket = atomicAdd(&p.tickets[r], 1u);
    __syncthreads();
    if (s_ticket != (unsigned)p.splits - 1) return;
    __threadfence();
    if (tid == 0) p.tickets[r] = 0;  // re-arm
    if (row >= p.G) return;
    // ---- row merge over the split partials (L2-resident)
    const float* pml = p.part_ml + (size_t)r * p.max_splits * 32;
    float MM = -INFINITY;
    for (int i = 0; i < p.splits; ++i) MM = fmaxf(MM, __ldcg(pml + i * 32 + row));
    float LL = 0.f;
#pragma unroll
    for (int j = 0; j < NCG; ++j) acc[j] = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int i = 0; i < p.splits; ++i) {
        const float mi_ = __ldcg(pml + i * 32 + row);
        const float wg = (MM == -INFINITY) ? 0.f : exp2f(mi_ - MM);
        LL += wg * __ldcg(pml + i * 32 + 16 + row);
        const float* po = p.part_O + ((size_t)(r * p.max_splits + i) * 16 + row) * D;
#pragma unroll
        for (int j = 0; j < NCG; ++j) {
            const float4 v = __ldcg(reinterpret_cast<const float4*>(po + cg * 4 + j * 32));
            acc[j].x += wg * v.x; acc[j].y += wg * v.y; acc[j].z += wg * v.z; acc[j].w += wg * v.w;
        }
    }
    store_out(acc, LL);
}

}  // namespace

int sparda_launch_attn(sparda_ctx* ctx, const void* Q, const void* pool, const int32_t* ids, int topk, int indexed,
                       int n_slots, void* O, cudaStream_t st) {
    const int D = ctx->cfg.head_dim;
    const uint64_t rows = (uint64_t)ctx->R * n_slots * 2 * S_BLK;
    const CUtensorMap* map;
    int rc = sparda_get_tmap(ctx, pool, rows, D, S_BLK, &map);
    if (rc) return rc;
    AttnParams p;
    p.Q = (const uint32_t*)Q;
    p.ids = ids;
    p.O = (__nv_bfloat16*)O;
    p.part_O = ctx->part_O;
    p.part_ml = ctx->part_ml;
    p.tickets = ctx->tickets + ctx->R;
    p.topk = topk;
    p.indexed = indexed;
    p.n_slots = n_slots;
    p.Hq = ctx->cfg.n_q_heads;
    p.Hkv = ctx->cfg.n_kv_heads;
    p.G = ctx->G;
    p.splits = sparda_resolve_splits(ctx, topk);
    p.max_splits = ctx->max_splits;
    p.scale_log2 = 1.4426950408889634f / sqrtf((float)D);
    dim3 grid(p.splits, ctx->R);
    static bool attr_set[2] = {false, false};
    if (D == 128) {
        if (!attr_set[0]) {
            SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(sparse_decode_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, AttnSmem<128>::TOTAL));
            attr_set[0] = true;
        }
        sparse_decode_kernel<128><<<grid, ATT_THREADS, AttnSmem<128>::TOTAL, st>>>(*map, p);
    } else {
        if (!attr_set[1]) {
            SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(sparse_decode_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, AttnSmem<64>::TOTAL));
            attr_set[1] = true;
        }
        sparse_decode_kernel<64><<<grid, ATT_THREADS, AttnSmem<64>::TOTAL, st>>>(*map, p);
    }
    SPARDA_CUDA_TRY(ctx, cudaGetLastError());
    ctx->launches++;
    return SPARDA_OK;
}
