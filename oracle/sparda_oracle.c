/*
 * sparda_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU restatement of what SparDA's decode-time hot path
 * computes, written from the paper text only (P:L<n> = /root/reference/PAPER.md line n).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call into this file.  It shares no code, header, table or helper with the CUDA path
 * under paper_2606_04511_b200/csrc/ and is never imported by it.
 *
 * Conventions: every tensor is row-major; "bf16" is the raw upper 16 bits of an IEEE fp32
 * (uint16_t); all sums are accumulated in double in ascending index order; every conversion
 * to bf16 is one round-to-nearest-even from the double value.  No blocking, fusion or
 * reordering beyond the definitions below.  OpenMP only splits the outermost loop over
 * independent (sequence, KV-head) units or query rows.
 *
 * Layouts (DESIGN.md "Readings" q11):
 *   kv     [R][Nb][2][S][D] bf16   R = B*Hkv rows, Nb blocks, plane 0 = K, plane 1 = V
 *   pool   [R][k ][2][S][D] bf16   slot i of row r holds block ids[r][i]
 *   Kpool  [R][Nb][D]       bf16   one mean-pooled key per block
 *   F      [R][D]           bf16   one Forecast head per GQA group
 *   Q      [B][Hq][D]       bf16   query head h belongs to group h / G
 *   ids    [R][k]           int32  ascending block ids, -1 padded
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): every function below is pinned by brute
 * force in an independent numpy/fp64 implementation, by invariants the paper fixes
 * (no-softmax claim P:L91, top-k = all blocks => dense attention) and by reduction to
 * torch.nn.functional.scaled_dot_product_attention.  The paper prints no worked numeric
 * example for this path.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

static double bf16_to_double(uint16_t h) {
    uint32_t u = ((uint32_t)h) << 16;
    float f;
    memcpy(&f, &u, 4);
    return (double)f;
}

/* One round-to-nearest-even from double to bf16 (8 significant bits, fp32 exponent range). */
static uint16_t double_to_bf16(double x) {
    if (isnan(x)) return 0x7FC0;
    uint16_t sign = signbit(x) ? 0x8000 : 0;
    double a = fabs(x);
    if (a == 0.0) return sign;
    if (isinf(a)) return sign | 0x7F80;
    int e;
    (void)frexp(a, &e); /* a = m * 2^e, m in [0.5, 1)  =>  floor(log2 a) = e - 1 */
    int p = e - 1;
    if (p < -126) p = -126;            /* subnormal range shares the quantum 2^-133 */
    double quantum = ldexp(1.0, p - 7); /* spacing of bf16 numbers in [2^p, 2^(p+1)) */
    double q = nearbyint(a / quantum);  /* default rounding mode = ties-to-even */
    double r = q * quantum;
    if (r >= ldexp(1.0, 128)) return sign | 0x7F80;
    float f = (float)r; /* exact: r has <= 8 significant bits */
    uint32_t u;
    memcpy(&u, &f, 4);
    return sign | (uint16_t)(u >> 16);
}

int sparda_oracle_threads(void) {
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void sparda_oracle_set_threads(int n) {
#ifdef _OPENMP
    extern void omp_set_num_threads(int);
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* helpers exported so the tests can pin the rounding itself */
uint16_t sparda_oracle_double_to_bf16(double x) { return double_to_bf16(x); }
double sparda_oracle_bf16_to_double(uint16_t h) { return bf16_to_double(h); }

/* o1 -- key compression, Eq.2 with kernel = stride = block size S (reading q1):
 *   Kpool[r,j,d] = bf16( (1/S) * sum_{t=0}^{S-1} K[r,j,t,d] )                                  */
void sparda_oracle_pool_keys(const uint16_t* kv, int64_t R, int64_t Nb, int S, int D, uint16_t* kpool) {
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < R; ++r)
        for (int64_t j = 0; j < Nb; ++j) {
            const uint16_t* Kblk = kv + ((r * Nb + j) * 2 + 0) * (int64_t)S * D;
            for (int d = 0; d < D; ++d) {
                double sum = 0.0;
                for (int t = 0; t < S; ++t) sum += bf16_to_double(Kblk[(int64_t)t * D + d]);
                kpool[(r * Nb + j) * D + d] = double_to_bf16(sum / (double)S);
            }
        }
}

/* o2 -- Forecast projection, Eq.3 (helper, not on the timed path):
 *   F[b, g, :] = bf16( X[b, :] . W_F[:, g*D:(g+1)*D] ),  W_F [hidden][Hkv*D]                     */
void sparda_oracle_forecast_project(const uint16_t* X, const uint16_t* WF, int64_t B, int64_t hidden, int Hkv,
                                    int D, uint16_t* F) {
    for (int64_t b = 0; b < B; ++b)
        for (int64_t c = 0; c < (int64_t)Hkv * D; ++c) {
            double sum = 0.0;
            for (int64_t i = 0; i < hidden; ++i)
                sum += bf16_to_double(X[b * hidden + i]) * bf16_to_double(WF[i * Hkv * D + c]);
            F[b * Hkv * D + c] = double_to_bf16(sum);
        }
}

/* o3 -- Forecast scoring, Eq.4, raw logits, no softmax, no scale:
 *   s[r,j] = sum_d F[r,d] * Kpool[r,j,d]      (double accumulate, rounded once to fp32)        */
void sparda_oracle_score(const uint16_t* F, const uint16_t* kpool, int64_t R, int64_t Nb, int D, float* scores) {
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < R; ++r)
        for (int64_t j = 0; j < Nb; ++j) {
            double sum = 0.0;
            for (int d = 0; d < D; ++d)
                sum += bf16_to_double(F[r * D + d]) * bf16_to_double(kpool[(r * Nb + j) * D + d]);
            scores[r * Nb + j] = (float)sum;
        }
}

typedef struct {
    float s;
    int32_t j;
} cand_t;

/* (score descending, index ascending) -- the lowest block index wins ties (reading q3) */
static int cand_cmp(const void* a, const void* b) {
    const cand_t* x = (const cand_t*)a;
    const cand_t* y = (const cand_t*)b;
    if (x->s > y->s) return -1;
    if (x->s < y->s) return 1;
    return (x->j > y->j) - (x->j < y->j);
}
static int int_cmp(const void* a, const void* b) {
    int32_t x = *(const int32_t*)a, y = *(const int32_t*)b;
    return (x > y) - (x < y);
}

/* f_top for one row: sort the n_cand candidates, keep the first min(k, n_cand), emit ascending ids,
 * pad with -1 (readings q4, q5).                                                                   */
static void topk_row(const float* s, int64_t n_cand, int k, int32_t* ids) {
    cand_t* c = (cand_t*)malloc(sizeof(cand_t) * (size_t)(n_cand > 0 ? n_cand : 1));
    for (int64_t j = 0; j < n_cand; ++j) {
        c[j].s = s[j];
        c[j].j = (int32_t)j;
    }
    qsort(c, (size_t)n_cand, sizeof(cand_t), cand_cmp);
    int64_t m = n_cand < k ? n_cand : k;
    for (int64_t i = 0; i < m; ++i) ids[i] = c[i].j;
    qsort(ids, (size_t)m, sizeof(int32_t), int_cmp);
    for (int64_t i = m; i < k; ++i) ids[i] = -1;
    free(c);
}

/* o4 -- f_top: top-k blocks of each row of s[R][Nb] among candidates [0, n_cand). */
void sparda_oracle_topk(const float* scores, int64_t R, int64_t Nb, int64_t n_cand, int k, int32_t* ids) {
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < R; ++r) topk_row(scores + r * Nb, n_cand, k, ids + r * k);
}

/* o5 -- prefetch, P:L306 (Alg.2 l.5): copy the selected blocks' K and V bytes to pool slots.
 * A slot whose id is -1 is left untouched.                                                         */
void sparda_oracle_gather(const uint16_t* kv, const int32_t* ids, int64_t R, int64_t Nb, int k, int S, int D,
                          uint16_t* pool) {
    const int64_t blk = 2 * (int64_t)S * D;
    for (int64_t r = 0; r < R; ++r)
        for (int i = 0; i < k; ++i) {
            int32_t j = ids[r * k + i];
            if (j < 0) continue;
            memcpy(pool + (r * k + i) * blk, kv + (r * Nb + j) * blk, (size_t)blk * 2);
        }
}

/* o6 -- block-sparse GQA attention with the real query, Eq.5 (Alg.2 l.7):
 *   for head h of sequence b, group g = h / G, row r = b*Hkv + g:
 *   z_t = (q_h . k_t) / sqrt(D) over every token t of every selected block (no causal mask, q7),
 *   p = softmax(z),  O_h = bf16( sum_t p_t v_t ).
 * pool_is_indexed = 0: slot i of `pool` ([R][k][2][S][D]) holds block ids[r][i]
 * pool_is_indexed = 1: `pool` is a full cache [R][n_slots][2][S][D] addressed by ids (layer 0)
 * A row with no valid id gives O = 0.  O_f64 (optional) receives the unrounded result.             */
void sparda_oracle_sparse_attn(const uint16_t* Q, const uint16_t* pool, const int32_t* ids, int pool_is_indexed,
                               int64_t B, int Hq, int Hkv, int D, int S, int k, int64_t n_slots, uint16_t* O,
                               double* O_f64) {
    const int G = Hq / Hkv;
    const int64_t blk = 2 * (int64_t)S * D;
    const double inv_sqrt_d = 1.0 / sqrt((double)D);
#pragma omp parallel for schedule(static)
    for (int64_t bh = 0; bh < B * Hq; ++bh) {
        const int64_t b = bh / Hq;
        const int h = (int)(bh % Hq);
        const int64_t r = b * Hkv + h / G;
        const uint16_t* q = Q + bh * D;
        double* z = (double*)malloc(sizeof(double) * (size_t)k * S);
        const uint16_t** vrow = (const uint16_t**)malloc(sizeof(uint16_t*) * (size_t)k * S);
        int64_t n = 0;
        for (int i = 0; i < k; ++i) {
            int32_t j = ids[r * k + i];
            if (j < 0) continue;
            const uint16_t* base = pool + (r * n_slots + (pool_is_indexed ? j : i)) * blk;
            for (int t = 0; t < S; ++t) {
                const uint16_t* kt = base + (int64_t)t * D;
                double dot = 0.0;
                for (int d = 0; d < D; ++d) dot += bf16_to_double(q[d]) * bf16_to_double(kt[d]);
                z[n] = dot * inv_sqrt_d;
                vrow[n] = base + (int64_t)S * D + (int64_t)t * D;
                ++n;
            }
        }
        double zmax = -INFINITY;
        for (int64_t t = 0; t < n; ++t)
            if (z[t] > zmax) zmax = z[t];
        double denom = 0.0;
        for (int64_t t = 0; t < n; ++t) {
            z[t] = exp(z[t] - zmax);
            denom += z[t];
        }
        for (int d = 0; d < D; ++d) {
            double acc = 0.0;
            for (int64_t t = 0; t < n; ++t) acc += (z[t] / denom) * bf16_to_double(vrow[t][d]);
            if (n == 0) acc = 0.0;
            O[bh * D + d] = double_to_bf16(acc);
            if (O_f64) O_f64[bh * D + d] = acc;
        }
        free(z);
        free(vrow);
    }
}

/* o7 -- dense attention over all Nb blocks of kv [R][Nb][2][S][D]; used by self-checks only. */
void sparda_oracle_dense_attn(const uint16_t* Q, const uint16_t* kv, int64_t B, int Hq, int Hkv, int D, int S,
                              int64_t Nb, uint16_t* O, double* O_f64) {
    const int G = Hq / Hkv;
    const double inv_sqrt_d = 1.0 / sqrt((double)D);
    const int64_t T = Nb * S;
#pragma omp parallel for schedule(static)
    for (int64_t bh = 0; bh < B * Hq; ++bh) {
        const int64_t r = (bh / Hq) * Hkv + (bh % Hq) / G;
        const uint16_t* q = Q + bh * D;
        double* z = (double*)malloc(sizeof(double) * (size_t)T);
        double zmax = -INFINITY;
        for (int64_t t = 0; t < T; ++t) {
            const uint16_t* kt = kv + ((r * Nb + t / S) * 2 + 0) * (int64_t)S * D + (t % S) * D;
            double dot = 0.0;
            for (int d = 0; d < D; ++d) dot += bf16_to_double(q[d]) * bf16_to_double(kt[d]);
            z[t] = dot * inv_sqrt_d;
            if (z[t] > zmax) zmax = z[t];
        }
        double denom = 0.0;
        for (int64_t t = 0; t < T; ++t) {
            z[t] = exp(z[t] - zmax);
            denom += z[t];
        }
        for (int d = 0; d < D; ++d) {
            double acc = 0.0;
            for (int64_t t = 0; t < T; ++t) {
                const uint16_t* vt = kv + ((r * Nb + t / S) * 2 + 1) * (int64_t)S * D + (t % S) * D;
                acc += (z[t] / denom) * bf16_to_double(vt[d]);
            }
            O[bh * D + d] = double_to_bf16(acc);
            if (O_f64) O_f64[bh * D + d] = acc;
        }
        free(z);
    }
}

/* o8 -- prefill selection with the Forecast indexer, P:L280 (Alg.1 l.2) + causal rule q8:
 * query position i may pick block j iff the block's last token <= i, i.e. n_cand(i) = (i+1)/S.
 *   F [Hkv][T][D], Kpool [Hkv][Nb][D]  ->  ids [Hkv][n_rows][k] for positions row0 .. row0+n_rows-1;
 *   scores_out (optional) [Hkv][n_rows][Nb] fp32 (entries j >= n_cand(i) are set to -inf).           */
void sparda_oracle_prefill_select(const uint16_t* F, const uint16_t* kpool, int Hkv, int64_t T, int64_t Nb, int D,
                                  int S, int64_t row0, int64_t n_rows, int k, int32_t* ids, float* scores_out) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t gi = 0; gi < (int64_t)Hkv * n_rows; ++gi) {
        const int64_t g = gi / n_rows;
        const int64_t i = row0 + gi % n_rows;
        int64_t n_cand = (i + 1) / S;
        if (n_cand > Nb) n_cand = Nb;
        float* s = (float*)malloc(sizeof(float) * (size_t)(Nb > 0 ? Nb : 1));
        const uint16_t* f = F + (g * T + i) * D;
        for (int64_t j = 0; j < n_cand; ++j) {
            double sum = 0.0;
            for (int d = 0; d < D; ++d) sum += bf16_to_double(f[d]) * bf16_to_double(kpool[(g * Nb + j) * D + d]);
            s[j] = (float)sum;
        }
        topk_row(s, n_cand, k, ids + gi * k);
        if (scores_out) {
            for (int64_t j = 0; j < Nb; ++j) scores_out[gi * Nb + j] = j < n_cand ? s[j] : -INFINITY;
        }
        free(s);
    }
}

/* o9 -- the comparison selector (InfLLM-V2 style; Eq.6 left term):
 *   S_shared[i,j] = sum_{h in group g} softmax_j( Q[h,i] . Kpool[g,j] / sqrt(D) ) over the causal
 *   candidates of row i, then the same f_top.     Q [Hq][T][D].                                      */
void sparda_oracle_prefill_select_baseline(const uint16_t* Q, const uint16_t* kpool, int Hq, int Hkv, int64_t T,
                                           int64_t Nb, int D, int S, int64_t row0, int64_t n_rows, int k,
                                           int32_t* ids, float* scores_out) {
    const int G = Hq / Hkv;
    const double inv_sqrt_d = 1.0 / sqrt((double)D);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t gi = 0; gi < (int64_t)Hkv * n_rows; ++gi) {
        const int64_t g = gi / n_rows;
        const int64_t i = row0 + gi % n_rows;
        int64_t n_cand = (i + 1) / S;
        if (n_cand > Nb) n_cand = Nb;
        double* shared = (double*)calloc((size_t)(Nb > 0 ? Nb : 1), sizeof(double));
        double* z = (double*)malloc(sizeof(double) * (size_t)(Nb > 0 ? Nb : 1));
        for (int hh = 0; hh < G; ++hh) {
            const uint16_t* q = Q + ((g * G + hh) * T + i) * D;
            double zmax = -INFINITY;
            for (int64_t j = 0; j < n_cand; ++j) {
                double sum = 0.0;
                for (int d = 0; d < D; ++d)
                    sum += bf16_to_double(q[d]) * bf16_to_double(kpool[(g * Nb + j) * D + d]);
                z[j] = sum * inv_sqrt_d;
                if (z[j] > zmax) zmax = z[j];
            }
            double denom = 0.0;
            for (int64_t j = 0; j < n_cand; ++j) {
                z[j] = exp(z[j] - zmax);
                denom += z[j];
            }
            for (int64_t j = 0; j < n_cand; ++j) shared[j] += z[j] / denom;
        }
        float* s = (float*)malloc(sizeof(float) * (size_t)(Nb > 0 ? Nb : 1));
        for (int64_t j = 0; j < n_cand; ++j) s[j] = (float)shared[j];
        topk_row(s, n_cand, k, ids + gi * k);
        if (scores_out)
            for (int64_t j = 0; j < Nb; ++j) scores_out[gi * Nb + j] = j < n_cand ? s[j] : -INFINITY;
        free(s);
        free(z);
        free(shared);
    }
}
