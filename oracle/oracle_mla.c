/*
 * oracle_mla.c -- TEST INFRASTRUCTURE, not the product.
 *
 * Plain, slow CPU reference for the mixed-step absorbed-MLA attention path
 * (paged latent cache append, decode rows, causal prefill-chunk rows).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 * It shares no code, header, table or constant with paper_2607_02043_b200/csrc/.
 *
 * What it follows.  PAPER.md never writes the attention math down ("The model and inference
 * kernels are unmodified", section 4.1); it names the model (DeepSeek-V2-Lite,
 * PAPER.md:377) and defines the mixed step as B decodes with K cached tokens each plus
 * prefill-chunk tokens in one batch (section 3.2) and chunked prefill as a
 * prompt processed in bounded chunks over steps (section 2.3).  The shapes
 * (16 heads, 512-d latent, 64-d RoPE key, scale 1/sqrt(192), page 64, bf16 in / fp32
 * accumulate, fp32 oracle) are fixed by BASELINE.json `north_star` / `configs[0]`; the
 * definition below is SURVEY.md section 8(c):
 *
 *   each cached token t stores c_t in R^512 and kR_t in R^64, shared by all heads;
 *   a query row (token j, head h) is q = [qC in R^512 | qR in R^64];
 *   s_t = sigma * (qC . c_t + qR . kR_t),  t = 0..n-1
 *   p   = softmax(s),  o = sum_t p_t c_t in R^512,  lse = ln sum_t exp(s_t)
 *   decode i: n = L_i (its own newest token is already in the cache, reading G2);
 *   chunk row j: n = P + j + 1 (prefix fully visible, self included, reading G3).
 *
 * The method reaches exactly this definition, so the oracle IS the definition written out:
 * two passes per row (scores buffered, max, then exp / sum / weighted sum), an explicit
 * page-table walk for every token (no gather into a contiguous buffer), fp32 arithmetic,
 * bf16 -> fp32 by `bits << 16`.  The 576-term dot product is a single loop that the compiler
 * may vectorise (`omp simd reduction`): the order of that fp32 sum is the only liberty taken.
 * oracle_dense_bruteforce is the same definition in double over a gathered, dense,
 * explicitly masked score matrix (tiny inputs only) and pins the walk/two-pass code above.
 *
 * Pins: tests/test_oracle_pins.py (closed forms, invariants, scipy/numpy dense softmax,
 * un-absorbed MLA identity).  Parity with real DeepSeek-V2-Lite activations or vLLM's kernel:
 * "parity unpinned" (no weights, no vLLM here; not required by north_star).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define H 16
#define DC 512
#define DR 64
#define D 576
#define PAGE 64

static inline float bf16_to_f32(uint16_t b) {
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, 4);
    return f;
}

static inline const uint16_t* token_row(const uint16_t* pool, const int32_t* page_table, int64_t t) {
    return pool + ((size_t)page_table[t / PAGE] * PAGE + (size_t)(t % PAGE)) * D;
}

/* a1: copy latent[n,512] | k_rope[n,64] into pool[page_table[pos/64]][pos%64][0:576]. */
int oracle_append(uint16_t* pool, int64_t num_pages, const uint16_t* latent, const uint16_t* k_rope,
                  int32_t n_tokens, const int32_t* page_table, int32_t table_len, int32_t start_pos) {
    if (n_tokens < 0 || start_pos < 0) return -1;
    for (int32_t j = 0; j < n_tokens; ++j) {
        int64_t pos = (int64_t)start_pos + j;
        if (pos / PAGE >= table_len) return -1;
        int32_t page = page_table[pos / PAGE];
        if (page < 0 || page >= num_pages) return -1;
        uint16_t* dst = pool + ((size_t)page * PAGE + (size_t)(pos % PAGE)) * D;
        memcpy(dst, latent + (size_t)j * DC, DC * sizeof(uint16_t));
        memcpy(dst + DC, k_rope + (size_t)j * DR, DR * sizeof(uint16_t));
    }
    return 0;
}

/* test helper: walk a page table and copy rows 0..n-1 out, [n,576]. */
int oracle_gather(const uint16_t* pool, const int32_t* page_table, int32_t n, uint16_t* out) {
    for (int64_t t = 0; t < n; ++t) memcpy(out + (size_t)t * D, token_row(pool, page_table, t), D * sizeof(uint16_t));
    return 0;
}

/* One query token (all 16 heads) over cache positions 0..n-1 of one sequence. */
static void attend_token(const uint16_t* pool, const int32_t* page_table, const uint16_t* q, int64_t n,
                         float sigma, float* out, float* lse, float* scores /* [16][n] */) {
    float qf[H][D];
    float kf[D];
    for (int h = 0; h < H; ++h)
        for (int d = 0; d < D; ++d) qf[h][d] = bf16_to_f32(q[h * D + d]);

    /* pass 1: scores, buffered */
    for (int64_t t = 0; t < n; ++t) {
        const uint16_t* row = token_row(pool, page_table, t);
        for (int d = 0; d < D; ++d) kf[d] = bf16_to_f32(row[d]);
        for (int h = 0; h < H; ++h) {
            float s = 0.0f;
#pragma omp simd reduction(+ : s)
            for (int d = 0; d < D; ++d) s += qf[h][d] * kf[d]; /* latent part, then rope part */
            scores[(size_t)h * n + t] = s * sigma;
        }
    }
    /* max */
    float m[H], l[H];
    for (int h = 0; h < H; ++h) {
        float mm = -INFINITY;
        for (int64_t t = 0; t < n; ++t) mm = fmaxf(mm, scores[(size_t)h * n + t]);
        m[h] = mm;
        l[h] = 0.0f;
    }
    /* pass 2: p = exp(s - m), l += p, acc += p * c_t */
    float acc[H][DC];
    memset(acc, 0, sizeof(acc));
    for (int64_t t = 0; t < n; ++t) {
        const uint16_t* row = token_row(pool, page_table, t);
        for (int d = 0; d < DC; ++d) kf[d] = bf16_to_f32(row[d]);
        for (int h = 0; h < H; ++h) {
            float p = expf(scores[(size_t)h * n + t] - m[h]);
            l[h] += p;
            for (int d = 0; d < DC; ++d) acc[h][d] += p * kf[d];
        }
    }
    for (int h = 0; h < H; ++h) {
        for (int d = 0; d < DC; ++d) out[h * DC + d] = acc[h][d] / l[h];
        if (lse) lse[h] = m[h] + logf(l[h]);
    }
}

/*
 * Generic rows entry: nq query tokens, token i attends positions 0..n_keys[i]-1 of the sequence
 * described by page_tables + seq_index[i]*table_stride.  out fp32 [nq,16,512], lse fp32 [nq,16] or NULL.
 */
int oracle_attend_rows(const uint16_t* pool, const int32_t* page_tables, int32_t table_stride,
                       const int32_t* seq_index, const uint16_t* q, int32_t nq, const int32_t* n_keys,
                       float sigma, float* out, float* lse) {
    int err = 0;
#pragma omp parallel
    {
        float* scores = NULL;
        size_t cap = 0;
#pragma omp for schedule(dynamic, 1)
        for (int32_t i = 0; i < nq; ++i) {
            int64_t n = n_keys[i];
            if (n < 1) { err = -1; continue; }
            if ((size_t)n * H > cap) {
                free(scores);
                cap = (size_t)n * H;
                scores = (float*)malloc(cap * sizeof(float));
            }
            const int32_t* pt = page_tables + (size_t)seq_index[i] * table_stride;
            attend_token(pool, pt, q + (size_t)i * H * D, n, sigma, out + (size_t)i * H * DC,
                         lse ? lse + (size_t)i * H : NULL, scores);
        }
        free(scores);
    }
    return err;
}

/*
 * The mixed step: n_dec decodes (one query token each over L_i cached tokens) plus one
 * causal chunk of chunk_len tokens over prefix_len cached tokens; the chunk's own tokens are already in
 * the cache (append precedes the step, reading G4).
 */
int oracle_mixed_step(const uint16_t* pool, int32_t n_dec, const uint16_t* q_dec,
                      const int32_t* dec_page_tables, int32_t dec_table_stride, const int32_t* dec_ctx_lens,
                      int32_t chunk_len, int32_t prefix_len, const uint16_t* q_chunk,
                      const int32_t* chunk_page_table, float sigma, float* out_dec, float* out_chunk,
                      float* lse_dec, float* lse_chunk) {
    int err = 0;
    if (n_dec > 0) {
        int32_t* idx = (int32_t*)malloc(sizeof(int32_t) * (size_t)n_dec);
        for (int32_t i = 0; i < n_dec; ++i) idx[i] = i;
        err |= oracle_attend_rows(pool, dec_page_tables, dec_table_stride, idx, q_dec, n_dec, dec_ctx_lens, sigma,
                                  out_dec, lse_dec);
        free(idx);
    }
    if (chunk_len > 0) {
        int32_t* idx = (int32_t*)calloc((size_t)chunk_len, sizeof(int32_t));
        int32_t* nk = (int32_t*)malloc(sizeof(int32_t) * (size_t)chunk_len);
        for (int32_t j = 0; j < chunk_len; ++j) nk[j] = prefix_len + j + 1;
        err |= oracle_attend_rows(pool, chunk_page_table, 0, idx, q_chunk, chunk_len, nk, sigma, out_chunk, lse_chunk);
        free(idx);
        free(nk);
    }
    return err;
}

/*
 * Dense brute force in double (tiny inputs): gather K[n_total,576], S = sigma * Q K^T with an explicit
 * boolean mask (row i sees t < n_keys[i]), row softmax, O = P K[:, :512].  probs [nq,16,n_total] returned
 * so "rows sum to 1" can be asserted.
 */
int oracle_dense_bruteforce(const uint16_t* pool, const int32_t* page_table, int32_t n_total, const uint16_t* q,
                            int32_t nq, const int32_t* n_keys, double sigma, double* out, double* probs) {
    double* K = (double*)malloc(sizeof(double) * (size_t)n_total * D);
    char* mask = (char*)malloc((size_t)nq * n_total);
    double* S = (double*)malloc(sizeof(double) * (size_t)n_total);
    for (int32_t t = 0; t < n_total; ++t) {
        const uint16_t* row = token_row(pool, page_table, t);
        for (int d = 0; d < D; ++d) K[(size_t)t * D + d] = (double)bf16_to_f32(row[d]);
    }
    for (int32_t i = 0; i < nq; ++i)
        for (int32_t t = 0; t < n_total; ++t) mask[(size_t)i * n_total + t] = (t < n_keys[i]);
    for (int32_t i = 0; i < nq; ++i) {
        for (int h = 0; h < H; ++h) {
            const uint16_t* qr = q + ((size_t)i * H + h) * D;
            double mx = -INFINITY;
            for (int32_t t = 0; t < n_total; ++t) {
                double s = 0.0;
                for (int d = 0; d < D; ++d) s += (double)bf16_to_f32(qr[d]) * K[(size_t)t * D + d];
                s *= sigma;
                if (!mask[(size_t)i * n_total + t]) s = -INFINITY;
                S[t] = s;
                if (s > mx) mx = s;
            }
            double sum = 0.0;
            for (int32_t t = 0; t < n_total; ++t) { S[t] = exp(S[t] - mx); sum += S[t]; }
            double* o = out + ((size_t)i * H + h) * DC;
            for (int d = 0; d < DC; ++d) o[d] = 0.0;
            for (int32_t t = 0; t < n_total; ++t) {
                double p = S[t] / sum;
                if (probs) probs[((size_t)i * H + h) * n_total + t] = p;
                for (int d = 0; d < DC; ++d) o[d] += p * K[(size_t)t * D + d];
            }
        }
    }
    free(K); free(mask); free(S);
    return 0;
}

int oracle_num_threads(void) {
    int n = 1;
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    n = omp_get_max_threads();
#endif
    return n;
}
