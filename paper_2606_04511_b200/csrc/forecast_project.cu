// Forecast projection (A4 / f4): F[b, g, :] = bf16( X[b, :] . W_F[:, g*D:(g+1)*D] ), Eq.3: the fourth per-layer
// projection, one Forecast head of width D per GQA group (4096 x 2 x 128 weights per layer = the 33.5 M added
// parameters of P:L95).  At decode this is a skinny GEMM, [B x hidden] x [hidden x Hkv*D], bound by reading W_F once (2 MiB
// for the 8B shape) and by latency: the whole thing should cost a few microseconds.
//
// One thread-block cluster per 64-column tile of W_F; the KS CTAs of a cluster split `hidden` between them (split-K).  A CTA
// stages its slab of W_F and the matching columns of X in shared memory (16-byte loads, rows padded by 16 bytes so that
// ldmatrix is conflict-free), 8 warps take one 8-column n-tile each and run mma.sync.m16n8k16 over up to 8 m-tiles of 16
// sequences (bf16 in, fp32 accumulate).  The split-K partials never touch global memory: every CTA sends its rows to the CTA
// of the cluster that owns them (st.shared::cluster), one cluster barrier, the owner adds the KS partials in rank order -- a
// fixed order, so the result is deterministic -- rounds once to bf16 and stores F.  (Round 1: 64 slab CTAs of FP32 FMAs, an
// L2 workspace and a last-CTA reduction: 52 us at batch 32.)
#include "sparda_internal.cuh"

namespace {

using namespace sparda;

constexpr int FP_THREADS = 256;
constexpr int FP_CT = 64;          // columns per cluster
constexpr int FP_MAX_ROWS = 128;   // sequences per pass (8 m-tiles)

struct FpParams {
    const uint16_t* X;   // [B][hidden]
    const uint16_t* W;   // [hidden][C]
    uint32_t* F;         // [B][C] as bf16 pairs
    int B, hidden, C;
    int ks;              // hidden rows per CTA (multiple of 16)
    int kc;              // rows staged per chunk (multiple of 16, <= 512)
    int rows_per;        // output rows owned by one CTA of the cluster, per pass
};

__device__ __forceinline__ void ldmatrix_x2_trans(uint32_t addr, uint32_t& r0, uint32_t& r1) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x2.trans.shared.b16 {%0,%1}, [%2];" : "=r"(r0), "=r"(r1) : "r"(addr));
}
__device__ __forceinline__ void cp_async_16(uint32_t smem_dst, const void* gsrc, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_dst), "l"(gsrc), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void fp_cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void fp_cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

__global__ void __launch_bounds__(FP_THREADS, 1) forecast_project_kernel(FpParams p) {
    extern __shared__ __align__(16) uint8_t fp_smem[];
    uint32_t KS, rank;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(KS));
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int gid = lane >> 2, tig = lane & 3;
    const int ctile = blockIdx.x / KS;
    const int col0 = ctile * FP_CT;
    const int k_begin = rank * p.ks;
    const int w_stride = FP_CT * 2 + 16;                 // bytes per staged W row
    const int x_stride = p.kc * 2 + 16;                  // bytes per staged X row
    uint8_t* Wt = fp_smem;
    uint8_t* Xs = Wt + (size_t)p.kc * w_stride;
    const int rows_cap = min(FP_MAX_ROWS, (p.B + 15) & ~15);
    float* red = reinterpret_cast<float*>(Xs + (size_t)rows_cap * x_stride);   // [KS][rows_per][FP_CT]
    fp_cluster_arrive();         // every CTA of the cluster is running before anyone writes a neighbour's shared memory
    pdl_wait();                  // X is the previous kernel's output in a model
    pdl_launch_dependents();
    bool cl_waited = false;

    for (int b0 = 0; b0 < p.B; b0 += FP_MAX_ROWS) {
        const int rows = min(FP_MAX_ROWS, p.B - b0);
        const int n_mt = (rows + 15) >> 4;
        float acc[FP_MAX_ROWS / 16][4];
#pragma unroll
        for (int mt = 0; mt < FP_MAX_ROWS / 16; ++mt) acc[mt][0] = acc[mt][1] = acc[mt][2] = acc[mt][3] = 0.f;
        for (int kc0 = 0; kc0 < p.ks; kc0 += p.kc) {
            const int kn = min(p.kc, p.ks - kc0);        // multiple of 16
            __syncthreads();                             // the previous chunk has been consumed
            // ---- stage W[k_begin + kc0 .. + kn)[col0 .. col0 + 64) and X[b0 .. b0 + rows)[same k range]
            // (cp.async: every 16-byte piece of the chunk is in flight at once -- one memory latency per chunk, no registers)
            {
                const int n_piece = kn * 8;              // 16-byte pieces of the W chunk
                const uint32_t wt_s = smem_u32(Wt), xs_s = smem_u32(Xs);
                for (int i = tid; i < n_piece; i += FP_THREADS)
                    cp_async_16(wt_s + (i >> 3) * w_stride + (i & 7) * 16, p.W + ((size_t)(k_begin + kc0 + (i >> 3)) * p.C + col0) + (i & 7) * 8, 16);
                const int ppr = kn / 8;                  // 16-byte pieces per X row
                const int n_xp = n_mt * 16 * ppr;
                for (int i = tid; i < n_xp; i += FP_THREADS) {
                    const int r = i / ppr, c = i % ppr;
                    const bool live = r < rows;          // rows beyond the batch are zero-filled (source size 0)
                    cp_async_16(xs_s + r * x_stride + c * 16, p.X + ((size_t)(b0 + (live ? r : 0)) * p.hidden + k_begin + kc0) + c * 8, live ? 16 : 0);
                }
                asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
            }
            __syncthreads();
            // ---- warp w: n-tile w (8 columns), all m-tiles
            const uint32_t wt_u32 = smem_u32(Wt) + (lane & 15) * w_stride + w * 16;
            const uint32_t xs_u32 = smem_u32(Xs) + ((lane & 7) + ((lane >> 3) & 1) * 8) * x_stride + (lane >> 4) * 16;
            for (int ks = 0; ks < kn / 16; ++ks) {
                uint32_t b0r, b1r;
                ldmatrix_x2_trans(wt_u32 + ks * 16 * w_stride, b0r, b1r);
#pragma unroll
                for (int mt = 0; mt < FP_MAX_ROWS / 16; ++mt) {
                    if (mt < n_mt) {
                        uint32_t a[4];
                        ldmatrix_x4(xs_u32 + mt * 16 * x_stride + ks * 32, a[0], a[1], a[2], a[3]);
                        mma_bf16_16816(acc[mt], a, b0r, b1r);
                    }
                }
            }
        }
        // ---- split-K reduction inside the cluster: rows [o * rows_per, (o + 1) * rows_per) of this pass belong to CTA o
        if (!cl_waited) { fp_cluster_wait(); cl_waited = true; }
        else { fp_cluster_arrive(); fp_cluster_wait(); }   // later passes: the owners have read the previous pass's partials
        const uint32_t red_u32 = smem_u32(red);
#pragma unroll
        for (int mt = 0; mt < FP_MAX_ROWS / 16; ++mt) {
            if (mt < n_mt) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int r = mt * 16 + h * 8 + gid;
                    if (r < rows) {
                        const uint32_t owner = (uint32_t)(r / p.rows_per), lr = (uint32_t)(r % p.rows_per);
                        uint32_t dst;
                        asm volatile("mapa.shared::cluster.u32 %0, %1, %2;"
                                     : "=r"(dst)
                                     : "r"(red_u32 + ((rank * p.rows_per + lr) * FP_CT + w * 8 + tig * 2) * 4), "r"(owner));
                        asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(dst), "f"(acc[mt][2 * h]), "f"(acc[mt][2 * h + 1]) : "memory");
                    }
                }
            }
        }
        fp_cluster_arrive();
        fp_cluster_wait();
        // ---- owner: add the KS partials in rank order, round once, store
        const int my_rows = min(p.rows_per, rows - (int)rank * p.rows_per);
        for (int e = tid; e < my_rows * (FP_CT / 2); e += FP_THREADS) {
            const int lr = e / (FP_CT / 2), c2 = e % (FP_CT / 2);
            float s0 = 0.f, s1 = 0.f;
            for (uint32_t q = 0; q < KS; ++q) {
                const float2 v = *reinterpret_cast<const float2*>(red + ((size_t)(q * p.rows_per + lr) * FP_CT + c2 * 2));
                s0 += v.x;
                s1 += v.y;
            }
            p.F[((size_t)(b0 + rank * p.rows_per + lr) * p.C + col0) / 2 + c2] = pack_bf16(s0, s1);
        }
    }
    if (!cl_waited) fp_cluster_wait();
}

}  // namespace

// (the split-K partials live in the cluster's shared memory: no workspace, any number of launches in flight)
int sparda_launch_forecast_project(sparda_ctx* ctx, const void* X, const void* WF, int hidden, void* F, cudaStream_t st) {
    FpParams p;
    p.X = (const uint16_t*)X;
    p.W = (const uint16_t*)WF;
    p.F = (uint32_t*)F;
    p.B = ctx->cfg.batch;
    p.hidden = hidden;
    p.C = ctx->cfg.n_kv_heads * ctx->cfg.head_dim;
    const int KS = hidden % 128 == 0 ? 8 : 4;                // hidden is a multiple of 64: ks stays a multiple of 16
    p.ks = hidden / KS;
    const int rows_cap = p.B >= FP_MAX_ROWS ? FP_MAX_ROWS : ((p.B + 15) & ~15);
    p.kc = p.ks < (rows_cap > 32 ? 256 : 512) ? p.ks : (rows_cap > 32 ? 256 : 512);
    p.rows_per = (rows_cap + KS - 1) / KS;
    const size_t smem = (size_t)p.kc * (FP_CT * 2 + 16) + (size_t)rows_cap * (p.kc * 2 + 16) + (size_t)KS * p.rows_per * FP_CT * sizeof(float);
    sparda_kernel_state& ks = ctx->kstate[SPARDA_K_PROJECT];
    if (!ks.attr_set) {
        SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(forecast_project_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        ks.attr_set = true;
    }
    if (smem > 200 * 1024) return SPARDA_EINVAL;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = KS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    at[1] = sparda_pdl_attr();
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((unsigned)(p.C / FP_CT * KS), 1, 1);
    lc.blockDim = dim3(FP_THREADS, 1, 1);
    lc.dynamicSmemBytes = smem;
    lc.stream = st;
    lc.attrs = at;
    lc.numAttrs = sparda_use_pdl(ctx) ? 2 : 1;
    SPARDA_CUDA_TRY(ctx, cudaLaunchKernelEx(&lc, forecast_project_kernel, p));
    ctx->launches++;
    return SPARDA_OK;
}
