// Forecast projection (A4 / f4): F[b, g, :] = bf16( X[b, :] . W_F[:, g*D:(g+1)*D] ), Eq.3: the fourth per-layer
// projection, one Forecast head of width D per GQA group (4096 x 2 x 128 weights per layer = the 33.5 M added
// parameters of P:L95).  At decode this is a GEMV per sequence and it is bound by streaming W_F once
// (hidden x Hkv*D x 2 bytes = 2 MiB for the 8B shape): split-K over `hidden` in slabs of 64 rows, one CTA per slab, every
// thread owns two adjacent output columns (4-byte loads, a warp reads 128 contiguous bytes of a weight row), the slab of
// X is staged in shared memory, fp32 accumulators for up to 32 sequences at a time.  Slab partials go to an L2-resident
// workspace; the last CTA (ticket) sums them in slab order -- a fixed order, so the result is deterministic -- and
// rounds once to bf16.
#include "sparda_internal.cuh"

namespace {

using namespace sparda;

constexpr int FP_SLAB = 64;     // rows of W_F per CTA
constexpr int FP_BT = 32;       // sequences accumulated per pass

__global__ void __launch_bounds__(256) forecast_project_kernel(const uint16_t* __restrict__ X, const uint32_t* __restrict__ W,
                                                                float* __restrict__ part, unsigned int* __restrict__ ticket,
                                                                uint32_t* __restrict__ F, int B, int hidden, int C /* Hkv * D */) {
    __shared__ float xs[FP_BT][FP_SLAB];
    __shared__ unsigned int s_last;
    const int slab = blockIdx.x, n_slabs = gridDim.x;
    const int C2 = C / 2;
    pdl_wait();                  // X is the previous kernel's output in a model
    pdl_launch_dependents();
    for (int b0 = 0; b0 < B; b0 += FP_BT) {
        const int nb = min(FP_BT, B - b0);
        __syncthreads();
        for (int e = threadIdx.x; e < nb * FP_SLAB; e += blockDim.x) {
            const int b = e / FP_SLAB, i = e % FP_SLAB;
            xs[b][i] = __uint_as_float((uint32_t)X[(size_t)(b0 + b) * hidden + slab * FP_SLAB + i] << 16);
        }
        __syncthreads();
        for (int c2 = threadIdx.x; c2 < C2; c2 += blockDim.x) {
            float a0[FP_BT], a1[FP_BT];
#pragma unroll
            for (int b = 0; b < FP_BT; ++b) a0[b] = a1[b] = 0.f;
            const uint32_t* wrow = W + (size_t)slab * FP_SLAB * C2 + c2;
#pragma unroll 4
            for (int i = 0; i < FP_SLAB; ++i) {
                const uint32_t w = __ldg(wrow + (size_t)i * C2);
                const float w0 = bf16_lo(w), w1 = bf16_hi(w);
#pragma unroll
                for (int b = 0; b < FP_BT; ++b)
                    if (b < nb) { a0[b] = fmaf(xs[b][i], w0, a0[b]); a1[b] = fmaf(xs[b][i], w1, a1[b]); }
            }
#pragma unroll
            for (int b = 0; b < FP_BT; ++b)
                if (b < nb) __stcg(reinterpret_cast<float2*>(part + ((size_t)slab * B + b0 + b) * C) + c2, make_float2(a0[b], a1[b]));
        }
    }
    // ---- the last CTA sums the slab partials in slab order and rounds
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(ticket, 1u) == (unsigned)n_slabs - 1 ? 1u : 0u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (threadIdx.x == 0) *ticket = 0;   // re-arm
    for (int e = threadIdx.x; e < B * C2; e += blockDim.x) {
        float s0 = 0.f, s1 = 0.f;
        for (int s = 0; s < n_slabs; ++s) {
            const float2 v = __ldcg(reinterpret_cast<const float2*>(part + (size_t)s * B * C) + e);
            s0 += v.x;
            s1 += v.y;
        }
        F[e] = pack_bf16(s0, s1);
    }
}

}  // namespace

int sparda_launch_forecast_project(sparda_ctx* ctx, const void* X, const void* WF, int hidden, void* F, int ws, cudaStream_t st) {
    const int C = ctx->cfg.n_kv_heads * ctx->cfg.head_dim;
    const int n_slabs = hidden / FP_SLAB;
    cudaLaunchAttribute at[1] = {sparda_pdl_attr()};
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3(n_slabs, 1, 1);
    lc.blockDim = dim3(256, 1, 1);
    lc.stream = st;
    lc.attrs = at;
    lc.numAttrs = sparda_use_pdl(ctx) ? 1 : 0;
    SPARDA_CUDA_TRY(ctx, cudaLaunchKernelEx(&lc, forecast_project_kernel, (const uint16_t*)X, (const uint32_t*)WF, ctx->fp_part + (size_t)ws * 128 * ctx->R * ctx->cfg.head_dim, ctx->fp_ticket + ws,
                                            (uint32_t*)F, ctx->cfg.batch, hidden, C));
    SPARDA_CUDA_TRY(ctx, cudaGetLastError());
    ctx->launches++;
    return SPARDA_OK;
}
