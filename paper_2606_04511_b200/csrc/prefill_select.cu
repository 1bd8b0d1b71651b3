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
// The per-row top-k is the real cost (plain ALU): 4 epilogue warps own one TMEM lane quadrant each, one thread per
// query row, and never leave registers except for a <= 24-entry boundary list:
//   pass 0   row min / max
//   7 passes bisection over 128 equal-width value buckets of [min, max]: count(s >= t) per pass (2 instr / element)
//   pass 8   collect the elements of the boundary bucket (value, id); exact k-th (value desc, id asc) among them
//   pass 9   emit ids with s > T or (s == T and id <= id_T) in ascending id order
// A row whose boundary bucket holds more than 24 elements (heavy ties) takes an exact bitwise radix search over
// order-preserving keys instead (33 passes; warp-uniform because tcgen05.ld is warp-collective).
// Scores never leave the SM.  a7' loops the same MMA over the G heads of the group, turns each head's accumulator
// into softmax probabilities (two TMEM passes) summed into an L2-resident per-CTA scratch tile, and runs the same
// selection on that tile.
#include "sparda_internal.cuh"

namespace {

using namespace sparda;

constexpr int PF_THREADS = 192;   // warp 0: TMA producer, warp 1: TMEM owner + MMA issuer, warps 2-5: epilogue
constexpr int PF_ROWS = 128;      // UMMA M
constexpr int PF_MAXN = 512;      // TMEM columns = max pooled keys per group
constexpr int PF_CAP = 24;        // boundary-list capacity per row
constexpr int PF_LIST_WORDS = 2 * PF_CAP;
constexpr int PF_WSTRIDE = 129;   // words between a thread's consecutive private words (bank-conflict free)
constexpr int PF_MAXK = 64;       // ids staged per row
constexpr int PF_OPITCH = PF_ROWS * 2 + 4;  // bytes between consecutive output positions (u16 per thread)
constexpr int PF_BUCKET_BITS = 7;

template <int D>
struct PfSmem {
    static constexpr int KH = D / 64;                            // 64-element (128 B) K slabs
    static constexpr int B_SLAB = PF_MAXN * 128;                 // one K slab of B: 512 rows x 128 B
    static constexpr int A_SLAB = PF_ROWS * 128;
    static constexpr int OFF_B = 0;
    static constexpr int OFF_A = OFF_B + KH * B_SLAB;
    static constexpr int OFF_LIST = OFF_A + KH * A_SLAB;
    static constexpr int OFF_OUT = OFF_LIST + PF_LIST_WORDS * PF_WSTRIDE * 4;
    static constexpr int OFF_STAT = OFF_OUT + PF_MAXK * PF_OPITCH;          // a7': (m, 1/l) per row, 1 KB
    static constexpr int OFF_BAR = (OFF_STAT + PF_ROWS * 8 + 7) & ~7;
    static constexpr int TOTAL = OFF_BAR + 64 + 1024;            // + slack for 1024-byte alignment
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

// Exact per-row top-k of src[0 .. ncand) for one thread's row; all 32 lanes of the warp call it together
// (loads are warp-collective), a lane with active == false only keeps the others company.
// On return the row's k ids (ascending) are staged as u16 at out_base[pos * PF_OPITCH].
template <class Src>
__device__ __forceinline__ void row_topk(const Src& src, int ncand, int nch, int k, bool active, uint32_t* list /* private, stride PF_WSTRIDE */,
                                         uint8_t* out_base) {
    float v[32];
    const float NEG = -INFINITY;
    if (!active) ncand = 0;
    // ---- pass 0: min / max over the candidates
    float lo = INFINITY, hi = -INFINITY;
    for (int c = 0; c < nch; ++c) {
        src.load(c, v);
#pragma unroll
        for (int e = 0; e < 32; ++e)
            if (c * 32 + e < ncand) { lo = fminf(lo, v[e]); hi = fmaxf(hi, v[e]); }
    }
    // ---- bisection over 2^7 equal-width buckets: largest bucket edge t_b with count(s >= t_b) >= k
    const float w = (hi - lo) * (1.0f / (1 << PF_BUCKET_BITS));
    int blo = 0, bhi = 1 << PF_BUCKET_BITS;          // count(s >= t_blo) >= k > count(s >= t_bhi);  t_128 = +inf
    int c_lo = ncand, c_hi = 0;
#pragma unroll 1
    for (int step = 0; step < PF_BUCKET_BITS; ++step) {
        const int mid = (blo + bhi) >> 1;
        const float t = fmaf((float)mid, w, lo);
        int cnt0 = 0, cnt1 = 0;
        for (int c = 0; c < nch; ++c) {
            src.load(c, v);
#pragma unroll
            for (int e = 0; e < 32; e += 2) {
                cnt0 += (c * 32 + e < ncand && v[e] >= t) ? 1 : 0;
                cnt1 += (c * 32 + e + 1 < ncand && v[e + 1] >= t) ? 1 : 0;
            }
        }
        const int cnt = cnt0 + cnt1;
        if (cnt >= k) { blo = mid; c_lo = cnt; } else { bhi = mid; c_hi = cnt; }
    }
    const float tlo = fmaf((float)blo, w, lo);
    const float thi = bhi == (1 << PF_BUCKET_BITS) ? INFINITY : fmaf((float)bhi, w, lo);
    const int need = k - c_hi;                        // how many of the boundary bucket are selected (>= 1)
    const bool slow = active && (c_lo - c_hi > PF_CAP);
    float T = NEG;                                    // k-th largest value
    int jT = -1;                                      // selected among s == T: ids <= jT
    bool general = false;                             // needs the tie-aware emission
    // ---- collect the boundary bucket and resolve it exactly
    {
        int n = 0;
        for (int c = 0; c < nch; ++c) {
            src.load(c, v);
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                const int j = c * 32 + e;
                if (j < ncand && v[e] >= tlo && v[e] < thi && n < PF_CAP) {
                    list[(2 * n) * PF_WSTRIDE] = __float_as_uint(v[e]);
                    list[(2 * n + 1) * PF_WSTRIDE] = (uint32_t)j;
                    ++n;
                }
            }
        }
        if (active && !slow) {
            // the need-th largest of the list by (value desc, position asc); the list is in ascending id order
            for (int e = 0; e < n; ++e) {
                const float se = __uint_as_float(list[(2 * e) * PF_WSTRIDE]);
                int rank = 0, later_eq = 0;
                for (int f = 0; f < n; ++f) {
                    const float sf = __uint_as_float(list[(2 * f) * PF_WSTRIDE]);
                    rank += (sf > se || (sf == se && f < e)) ? 1 : 0;
                    later_eq += (sf == se && f > e) ? 1 : 0;
                }
                if (rank == need - 1) {
                    T = se;
                    jT = (int)list[(2 * e + 1) * PF_WSTRIDE];
                    general = later_eq > 0;           // an equal element with a larger id stays out
                }
            }
        }
    }
    // ---- heavy ties: exact bitwise search of the k-th largest order-preserving key (warp-uniform)
    int need_eq = 0;
    if (__any_sync(0xffffffffu, slow)) {
        uint32_t tk = 0;
#pragma unroll 1
        for (int bit = 31; bit >= 0; --bit) {
            const uint32_t cand = tk | (1u << bit);
            int cnt = 0;
            for (int c = 0; c < nch; ++c) {
                src.load(c, v);
#pragma unroll
                for (int e = 0; e < 32; ++e) cnt += (c * 32 + e < ncand && orderable(v[e] + 0.0f) >= cand) ? 1 : 0;
            }
            if (cnt >= k) tk = cand;
        }
        int cgt = 0;
        for (int c = 0; c < nch; ++c) {
            src.load(c, v);
#pragma unroll
            for (int e = 0; e < 32; ++e) cgt += (c * 32 + e < ncand && orderable(v[e] + 0.0f) > tk) ? 1 : 0;
        }
        if (slow) { T = key_to_float(tk); need_eq = k - cgt; general = true; }
    }
    // ---- emit ascending ids
    int pos = 0;
    if (__any_sync(0xffffffffu, general)) {
        int eq_seen = 0;
        for (int c = 0; c < nch; ++c) {
            src.load(c, v);
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                const int j = c * 32 + e;
                if (j < ncand) {
                    bool sel = v[e] > T;
                    if (v[e] == T) {
                        sel = slow ? (eq_seen < need_eq) : (j <= jT);
                        ++eq_seen;
                    }
                    if (sel && pos < PF_MAXK) { *reinterpret_cast<uint16_t*>(out_base + pos * PF_OPITCH) = (uint16_t)j; ++pos; }
                }
            }
        }
    } else {
        for (int c = 0; c < nch; ++c) {
            src.load(c, v);
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                const int j = c * 32 + e;
                if (j < ncand && v[e] >= T && pos < PF_MAXK) { *reinterpret_cast<uint16_t*>(out_base + pos * PF_OPITCH) = (uint16_t)j; ++pos; }
            }
        }
    }
}

template <int D, bool BASELINE>
__global__ void __launch_bounds__(PF_THREADS, 1)
prefill_select_kernel(const __grid_constant__ CUtensorMap tmapA, const __grid_constant__ CUtensorMap tmapB, PfParams p) {
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
        mbar_init(tmem_empty, 4);
        mbar_fence_init();
        fence_proxy_async_smem();
        tma_prefetch_desc(&tmapA);
        tma_prefetch_desc(&tmapB);
    }
    if (warp == 1) tmem_alloc(tmem_slot, PF_MAXN);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    // Tile schedule (identical in every role): tiles sorted by cost (descending row index), dealt in a snake over the
    // group's CTAs.  Tile s covers rows [m0, m0 + 128), m0 = (mt_lo + n_tiles - 1 - s) * 128.
    auto tile_of_round = [&](int r) -> int {
        const int s = r * n_cta + ((r & 1) ? (n_cta - 1 - cta) : cta);
        return s < p.n_tiles ? (p.mt_lo + p.n_tiles - 1 - s) : -1;
    };
    const int n_rounds = (p.n_tiles + n_cta - 1) / n_cta;
    auto tile_ncols = [&](int mt) -> int { return min(p.n_blocks, (mt * PF_ROWS + PF_ROWS) / 64); };  // visible blocks of the tile's last row

    if (warp == 0) {
        // =============================== TMA producer ===============================
        if (lane == 0) {
            const int nb_boxes = (p.n_blocks + 255) / 256;
            mbar_arrive_expect_tx(b_full, (uint32_t)(KH * nb_boxes * 256 * 128));
            for (int kh = 0; kh < KH; ++kh)
                for (int nh = 0; nh < nb_boxes; ++nh)
                    tma_load_2d(smem + SM::OFF_B + kh * SM::B_SLAB + nh * 256 * 128, &tmapB, kh * 64, g * p.n_blocks + nh * 256, b_full);
            uint32_t it = 0;
            for (int r = 0; r < n_rounds; ++r) {
                const int mt = tile_of_round(r);
                if (mt < 0 || tile_ncols(mt) <= p.topk) continue;   // nothing to rank: every candidate is selected
                for (int h = 0; h < NH; ++h, ++it) {
                    mbar_wait(a_empty, (it & 1) ^ 1);
                    mbar_arrive_expect_tx(a_full, (uint32_t)(KH * SM::A_SLAB));
                    const int arow = (BASELINE ? (g * p.G + h) : g) * p.T + mt * PF_ROWS;
                    for (int kh = 0; kh < KH; ++kh) tma_load_2d(smem + SM::OFF_A + kh * SM::A_SLAB, &tmapA, kh * 64, arow, a_full);
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
                    mbar_wait(a_full, it & 1);
                    mbar_wait(tmem_empty, (it & 1) ^ 1);
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
        // =============================== epilogue: one thread per query row ===============================
        const int q = warp & 3;                                  // TMEM lane quadrant this warp may access
        const int trow = q * 32 + lane;                          // row within the tile
        uint32_t* list = reinterpret_cast<uint32_t*>(smem + SM::OFF_LIST) + trow;
        uint8_t* out_base = smem + SM::OFF_OUT + trow * 2;
        float2* stat = reinterpret_cast<float2*>(smem + SM::OFF_STAT) + trow;
        float* scr = BASELINE ? p.scratch + (size_t)blockIdx.x * PF_MAXN * PF_ROWS + trow : nullptr;
        const TmemRow trsrc{tmem_base + ((uint32_t)(q * 32) << 16)};
        uint32_t it = 0;
        for (int r = 0; r < n_rounds; ++r) {
            const int mt = tile_of_round(r);
            if (mt < 0) continue;
            const int i = mt * PF_ROWS + trow;                   // query position of this thread
            const bool in_chunk = i >= p.row0 && i < p.row0 + p.n_rows;
            const int ncand = min(p.n_blocks, (i + 1) / 64);
            int32_t* dst = p.ids + ((size_t)g * p.n_rows + (i - p.row0)) * p.topk;
            const int ncols = tile_ncols(mt);
            if (ncols <= p.topk) {                               // whole tile: every candidate is selected (reading q5)
                if (in_chunk)
                    for (int s = 0; s < p.topk; ++s) dst[s] = s < ncand ? s : -1;
                continue;
            }
            const int wmax = min(p.n_blocks, (mt * PF_ROWS + q * 32 + 32) / 64);   // candidates of the warp's last row
            const int nch = (wmax + 31) / 32;
            const bool ranked = in_chunk && ncand > p.topk;
            if (BASELINE) {
                // a7': per head, softmax over the causal candidates of the row, summed into the scratch tile
                float v[32];
                for (int h = 0; h < NH; ++h, ++it) {
                    mbar_wait(mma_done, it & 1);
                    tc_fence_after();
                    float m = -INFINITY;
                    for (int c = 0; c < nch; ++c) {
                        trsrc.load(c, v);
#pragma unroll
                        for (int e = 0; e < 32; ++e)
                            if (c * 32 + e < ncand) m = fmaxf(m, v[e]);
                    }
                    const float ms = m * p.scale_log2;
                    float l = 0.f;
                    for (int c = 0; c < nch; ++c) {
                        trsrc.load(c, v);
#pragma unroll
                        for (int e = 0; e < 32; ++e)
                            if (c * 32 + e < ncand) l += exp2f(fmaf(v[e], p.scale_log2, -ms));
                    }
                    const float inv = ncand > 0 ? 1.0f / l : 0.f;
                    for (int c = 0; c < nch; ++c) {
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
                (void)stat;
                if (__any_sync(0xffffffffu, ranked)) row_topk(ScratchRow{scr}, ncand, nch, p.topk, ranked, list, out_base);
            } else {
                mbar_wait(mma_done, it & 1);
                ++it;
                tc_fence_after();
                if (__any_sync(0xffffffffu, ranked)) row_topk(trsrc, ncand, nch, p.topk, ranked, list, out_base);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tmem_empty);
            }
            if (ranked) {
                if ((p.topk & 3) == 0) {
                    for (int s = 0; s < p.topk; s += 4) {
                        int4 o;
                        o.x = *reinterpret_cast<const uint16_t*>(out_base + (s + 0) * PF_OPITCH);
                        o.y = *reinterpret_cast<const uint16_t*>(out_base + (s + 1) * PF_OPITCH);
                        o.z = *reinterpret_cast<const uint16_t*>(out_base + (s + 2) * PF_OPITCH);
                        o.w = *reinterpret_cast<const uint16_t*>(out_base + (s + 3) * PF_OPITCH);
                        *reinterpret_cast<int4*>(dst + s) = o;
                    }
                } else {
                    for (int s = 0; s < p.topk; ++s) dst[s] = *reinterpret_cast<const uint16_t*>(out_base + s * PF_OPITCH);
                }
            } else if (in_chunk) {
                for (int s = 0; s < p.topk; ++s) dst[s] = s < ncand ? s : -1;
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, PF_MAXN);
    }
}

template <int D, bool BASELINE>
int launch(sparda_ctx* ctx, const void* A, const void* Kpool, int T, int n_blocks, int row0, int n_rows, int topk, int32_t* ids,
           cudaStream_t st) {
    using SM = PfSmem<D>;
    const int Hkv = ctx->cfg.n_kv_heads, G = ctx->G;
    const CUtensorMap *mapA, *mapB;
    int rc = sparda_get_tmap(ctx, A, (uint64_t)(BASELINE ? Hkv * G : Hkv) * T, D, PF_ROWS, &mapA);
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
    p.mt_lo = row0 / PF_ROWS;
    p.n_tiles = (row0 + n_rows + PF_ROWS - 1) / PF_ROWS - p.mt_lo;
    if (per_group > p.n_tiles) per_group = p.n_tiles;
    p.scale_log2 = 1.4426950408889634f / sqrtf((float)D);
    p.scratch = nullptr;
    if (BASELINE) p.scratch = ctx->pf_scratch;
    static bool attr_set = false;
    if (!attr_set) {
        SPARDA_CUDA_TRY(ctx, cudaFuncSetAttribute(prefill_select_kernel<D, BASELINE>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM::TOTAL));
        attr_set = true;
    }
    prefill_select_kernel<D, BASELINE><<<per_group * Hkv, PF_THREADS, SM::TOTAL, st>>>(*mapA, *mapB, p);
    SPARDA_CUDA_TRY(ctx, cudaGetLastError());
    ctx->launches++;
    return SPARDA_OK;
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
