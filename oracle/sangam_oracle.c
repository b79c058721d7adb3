/*
 * sangam_oracle.c -- plain, slow, fp64 CPU oracle for the Sangam hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares
 * no code, header, table or helper with the CUDA library under
 * paper_2607_04206_b200/csrc/ and neither includes the other.
 *
 * What it computes is the plain DEFINITION of the path (the method -- tiling, online
 * softmax, split-KV -- is a re-association of this one sum, so the oracle is the
 * definition written out, not an algorithm to mimic):
 *
 *   - oracle_kv_write: scatter fresh K/V rows into 16-token pages
 *       (PagedAttention with page size 16; the cache is
 *        recomputed at block boundaries and reused inside a block).
 *   - oracle_block_attn: unmasked, bidirectional softmax attention of every query row
 *       of a request over that request's whole paged context
 *       ("the causal mask is dropped so tokens attend bidirectionally over the full
 *        prompt-and-response"; a decode "contributes an entire response
 *        block while attending over the prompt and response context", PAPER.md:33;
 *        GQA for Dream-7B, MHA for LLaDA-8B).
 *   - oracle_attn_contiguous: the same definition over per-request contiguous K/V
 *       (a second, independent addressing; pins the paged one).
 *
 * Readings of points the paper is silent on are DESIGN.md "Readings" S1-S18
 * (q head h uses kv head h / G; slot = page*16 + offset; slot < 0 skipped;
 * c_r = 0 gives zero rows; no mask, bias or soft-cap).
 *
 * Pins: tests/test_oracle_pins.py (-m "not gpu") checks every function here against
 * closed forms, invariants, a dense numpy softmax(QK^T)V and brute force on tiny inputs.
 *
 * Arithmetic: inputs are bf16 bit patterns widened exactly to double; `scale` is the
 * float32 handed to the GPU, widened; everything else is double.  Plain loops, no
 * blocking, no reordering.  OpenMP only distributes independent (row, head) pairs.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PAGE 16

static inline double bf16_to_f64(uint16_t b) {
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* k, v: uint16 [T_new][Hkv][D]; pools: uint16 [P][Hkv][16][D]; 16-bit copies, no FP. */
int oracle_kv_write(const uint16_t* k, const uint16_t* v, const int32_t* slot_mapping,
                    int32_t num_tokens, int32_t Hkv, int32_t D,
                    uint16_t* k_pages, uint16_t* v_pages) {
    for (int32_t i = 0; i < num_tokens; ++i) {
        int32_t s = slot_mapping[i];
        if (s < 0) continue;                       /* graph padding (reading S10) */
        int64_t page = s / ORACLE_PAGE, off = s % ORACLE_PAGE;
        for (int32_t h = 0; h < Hkv; ++h)
            for (int32_t d = 0; d < D; ++d) {
                int64_t dst = ((page * Hkv + h) * ORACLE_PAGE + off) * D + d;
                int64_t src = ((int64_t)i * Hkv + h) * D + d;
                k_pages[dst] = k[src];
                v_pages[dst] = v[src];
            }
    }
    return 0;
}

/*
 * Paged attention, the definition:
 *   for request r, query row t, q head h, g = h / G:
 *     s[j]   = scale * sum_d q[t][h][d] * K[page(j)][g][j%16][d]      j < c_r
 *     m      = max_j s[j];  p[j] = exp(s[j] - m);  l = sum_j p[j]
 *     out[d] = (sum_j p[j] * V[page(j)][g][j%16][d]) / l
 *     lse    = m + log l
 * row_sel == NULL: every row of the batch, out is [T_q][Hq][D].
 * row_sel != NULL: only the n_sel listed global row indices, out is [n_sel][Hq][D].
 * lse, rowsum may be NULL.  Pages are indexed directly through block_table.
 */
int oracle_block_attn(const uint16_t* q, const uint16_t* k_pages, const uint16_t* v_pages,
                      const int32_t* block_table, int32_t W,
                      const int32_t* cu_q_lens, const int32_t* ctx_lens, int32_t R,
                      int32_t Hq, int32_t Hkv, int32_t D, float scale_f32,
                      const int32_t* row_sel, int32_t n_sel,
                      double* out, double* lse, double* rowsum) {
    if (Hkv <= 0 || Hq % Hkv != 0) return -1;
    const int32_t G = Hq / Hkv;
    const double scale = (double)scale_f32;
    const int32_t total_q = cu_q_lens[R];
    const int64_t n_rows = row_sel ? n_sel : total_q;
    int32_t max_c = 0;
    for (int32_t r = 0; r < R; ++r) if (ctx_lens[r] > max_c) max_c = ctx_lens[r];

#pragma omp parallel
    {
        double* s = (double*)malloc(sizeof(double) * (size_t)(max_c > 0 ? max_c : 1));
        double* acc = (double*)malloc(sizeof(double) * (size_t)D);
#pragma omp for schedule(dynamic, 1) collapse(2)
        for (int64_t i = 0; i < n_rows; ++i) {
            for (int32_t h = 0; h < Hq; ++h) {
                const int32_t t = row_sel ? row_sel[i] : (int32_t)i;
                int32_t r = 0;
                while (r < R && !(cu_q_lens[r] <= t && t < cu_q_lens[r + 1])) ++r;
                double* o = out + ((int64_t)i * Hq + h) * D;
                if (r >= R || ctx_lens[r] <= 0) {               /* reading S13 */
                    for (int32_t d = 0; d < D; ++d) o[d] = 0.0;
                    if (lse) lse[i * Hq + h] = -INFINITY;
                    if (rowsum) rowsum[i * Hq + h] = 0.0;
                    continue;
                }
                const int32_t c = ctx_lens[r];
                const int32_t g = h / G;                          /* reading S4 */
                const uint16_t* qrow = q + ((int64_t)t * Hq + h) * D;
                double m = -INFINITY;
                for (int32_t j = 0; j < c; ++j) {
                    const int64_t page = block_table[(int64_t)r * W + j / ORACLE_PAGE];
                    const uint16_t* krow = k_pages + ((page * Hkv + g) * ORACLE_PAGE + j % ORACLE_PAGE) * D;
                    double dot = 0.0;
                    for (int32_t d = 0; d < D; ++d) dot += bf16_to_f64(qrow[d]) * bf16_to_f64(krow[d]);
                    s[j] = scale * dot;
                    if (s[j] > m) m = s[j];
                }
                double l = 0.0;
                for (int32_t d = 0; d < D; ++d) acc[d] = 0.0;
                for (int32_t j = 0; j < c; ++j) {
                    const double p = exp(s[j] - m);
                    l += p;
                    const int64_t page = block_table[(int64_t)r * W + j / ORACLE_PAGE];
                    const uint16_t* vrow = v_pages + ((page * Hkv + g) * ORACLE_PAGE + j % ORACLE_PAGE) * D;
                    for (int32_t d = 0; d < D; ++d) acc[d] += p * bf16_to_f64(vrow[d]);
                }
                for (int32_t d = 0; d < D; ++d) o[d] = acc[d] / l;
                if (lse) lse[i * Hq + h] = m + log(l);
                if (rowsum) {
                    double rs = 0.0;
                    for (int32_t j = 0; j < c; ++j) rs += exp(s[j] - m) / l;
                    rowsum[i * Hq + h] = rs;
                }
            }
        }
        free(s);
        free(acc);
    }
    return 0;
}

/*
 * Same definition over contiguous per-request K/V: k, v are uint16 [sum_r c_r][Hkv][D],
 * request r owning rows cu_ctx[r] .. cu_ctx[r+1]-1.  No pages, no block table.
 */
int oracle_attn_contiguous(const uint16_t* q, const uint16_t* k, const uint16_t* v,
                           const int64_t* cu_ctx, const int32_t* cu_q_lens, int32_t R,
                           int32_t Hq, int32_t Hkv, int32_t D, float scale_f32, double* out) {
    if (Hkv <= 0 || Hq % Hkv != 0) return -1;
    const int32_t G = Hq / Hkv;
    const double scale = (double)scale_f32;
    for (int32_t r = 0; r < R; ++r) {
        const int64_t c = cu_ctx[r + 1] - cu_ctx[r];
        double* s = (double*)malloc(sizeof(double) * (size_t)(c > 0 ? c : 1));
        for (int32_t t = cu_q_lens[r]; t < cu_q_lens[r + 1]; ++t)
            for (int32_t h = 0; h < Hq; ++h) {
                double* o = out + ((int64_t)t * Hq + h) * D;
                for (int32_t d = 0; d < D; ++d) o[d] = 0.0;
                if (c <= 0) continue;
                const int32_t g = h / G;
                double m = -INFINITY;
                for (int64_t j = 0; j < c; ++j) {
                    double dot = 0.0;
                    for (int32_t d = 0; d < D; ++d)
                        dot += bf16_to_f64(q[((int64_t)t * Hq + h) * D + d]) *
                               bf16_to_f64(k[((cu_ctx[r] + j) * Hkv + g) * D + d]);
                    s[j] = scale * dot;
                    if (s[j] > m) m = s[j];
                }
                double l = 0.0;
                for (int64_t j = 0; j < c; ++j) { s[j] = exp(s[j] - m); l += s[j]; }
                for (int64_t j = 0; j < c; ++j)
                    for (int32_t d = 0; d < D; ++d)
                        o[d] += s[j] * bf16_to_f64(v[((cu_ctx[r] + j) * Hkv + g) * D + d]);
                for (int32_t d = 0; d < D; ++d) o[d] /= l;
            }
        free(s);
    }
    return 0;
}

/*
 * Split-KV merge, step a9: partial i holds the UNNORMALISED sum
 * O_i = sum_j exp(s_j - m_i) v_j, its max m_i and its sum l_i.
 *   m* = max_i m_i;  l* = sum_i l_i e^{m_i - m*};  O* = sum_i O_i e^{m_i - m*};  out = O* / l*
 */
int oracle_combine(const double* O_parts, const double* m_parts, const double* l_parts,
                   int32_t n_parts, int32_t D, double* out) {
    double ms = -INFINITY, ls = 0.0;
    for (int32_t i = 0; i < n_parts; ++i) if (m_parts[i] > ms) ms = m_parts[i];
    for (int32_t d = 0; d < D; ++d) out[d] = 0.0;
    if (ms == -INFINITY) return 0;
    for (int32_t i = 0; i < n_parts; ++i) {
        if (m_parts[i] == -INFINITY) continue;
        const double w = exp(m_parts[i] - ms);
        ls += l_parts[i] * w;
        for (int32_t d = 0; d < D; ++d) out[d] += O_parts[(int64_t)i * D + d] * w;
    }
    for (int32_t d = 0; d < D; ++d) out[d] /= ls;
    return 0;
}
