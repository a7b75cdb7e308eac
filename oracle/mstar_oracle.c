/*
 * mstar_oracle.c -- CPU ORACLE for attention over a paged KV cache.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the plain, slow, fp64 definition the CUDA path is checked against.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it; the
 * product (paper_2606_12688_b200/) never does and shares no code, header, table or helper with it.
 *
 * What it computes (the paper gives no formula of its own -- its attention is a FlashInfer library
 * call, sec. 3.3 and :430 App. I, over "a single paged KV pool ... reading page tables
 * in place", PAPER.md:198 -- so the definition is the textbook one):
 *
 *   GATHER(s):  K_s[j] = k_pool[block_table[s][j div p]][:, j mod p, :],  j = 0 .. L_s-1  (same for V)
 *   DECODE:     x_j = scale * sum_d q[s][h][d] * K_s[j][h div G][d]
 *               M = max_j x_j;  w_j = exp(x_j - M);  Z = sum_j w_j
 *               out[s][h][:] = (sum_j w_j V_s[j][h div G][:]) / Z;   lse[s][h] = M + ln Z
 *   PREFILL:    the same for query row i of sequence s restricted to j <= P_s + i, P_s = L_s - n_s
 *               (bottom-right aligned causal mask, "causal masking over a cached prefix",
 *               BASELINE.json north_star; reading R6)
 *   APPEND:     pool[slot div p][h][slot mod p][:] = new[t][h][:] as 16-bit words; slot < 0 skipped
 *   GATHER (as an operation of its own) and COPY_PAGES (the page moves behind
 *               "paging, offload, by-reference transfer", and prefill/decode disaggregation, :116):
 *               out[cu[s] + j][h][:] = pool[block_table[s][j div p]][h][j mod p][:];
 *               dst_pool[dst_pages[i]] = src_pool[src_pages[i]] (all heads and slots), in order of i, id < 0 skipped
 *   COMBINE:    M = max_i m_i; out = sum_i e^{m_i-M} O_i / sum_i e^{m_i-M} l_i; lse = M + ln(sum_i ...)
 *               (split-K merge, BASELINE.json north_star "log-sum-exp combine pass")
 *
 * All arithmetic is fp64 on the exact values of the bf16 inputs (bf16 -> fp64 is exact); no tiling,
 * no online softmax, no reordering: every loop is the formula above written out.  OpenMP only
 * distributes independent (row, head) outputs over threads.
 *
 * Pins (tests/test_oracle_pins.py, all run without a GPU): brute-force numpy softmax(QK^T)V on dense
 * gathered K/V; closed forms (L=1 => V row; q=0 => mean of V rows; V==1 => 1; two-key logistic);
 * rows of P sum to 1; page-id permutation invariance; shared-prefix == duplicated-prefix; shift
 * invariance; split + COMBINE == unsplit; prefill n=1 == decode; last prefill row == decode;
 * causality under +-1e30 poisoning of future keys; chunked prefill identity.  No function here is
 * "parity unpinned".
 *
 * Pool layout: [num_pages][Hkv][p][D] uint16 (bf16 bit patterns), K and V separate.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static double bf16_to_f64(uint16_t b) {
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

/* APPEND: bit copy of 16-bit words, sequential in t so that "last writer wins" (R19). */
void oracle_kv_append(uint16_t* k_pool, uint16_t* v_pool, int32_t Hkv, int32_t p, int32_t D,
                      const uint16_t* k_new, const uint16_t* v_new, const int64_t* slot_mapping,
                      int64_t T) {
    for (int64_t t = 0; t < T; ++t) {
        int64_t s = slot_mapping[t];
        if (s < 0) continue;
        int64_t page = s / p, off = s % p;
        for (int32_t h = 0; h < Hkv; ++h) {
            size_t dst = (((size_t)page * Hkv + h) * p + off) * D;
            size_t src = ((size_t)t * Hkv + h) * D;
            for (int32_t d = 0; d < D; ++d) {
                k_pool[dst + d] = k_new[src + d];
                v_pool[dst + d] = v_new[src + d];
            }
        }
    }
}

/* GATHER: contiguous fp64 K_s, V_s of shape [L][Hkv][D] for one sequence. */
void oracle_gather(double* K, double* V, const uint16_t* k_pool, const uint16_t* v_pool,
                   const int32_t* block_table_row, int32_t L, int32_t Hkv, int32_t p, int32_t D) {
    for (int32_t j = 0; j < L; ++j) {
        int64_t page = block_table_row[j / p];
        int32_t off = j % p;
        for (int32_t h = 0; h < Hkv; ++h) {
            size_t src = (((size_t)page * Hkv + h) * p + off) * D;
            size_t dst = ((size_t)j * Hkv + h) * D;
            for (int32_t d = 0; d < D; ++d) {
                K[dst + d] = bf16_to_f64(k_pool[src + d]);
                V[dst + d] = bf16_to_f64(v_pool[src + d]);
            }
        }
    }
}

/* One attention row over keys 0 .. n_keys-1 of kv head g.  probs (optional) receives w_j / Z. */
static void attend_row(double* out, double* lse, double* probs, const uint16_t* q_row,
                       const double* K, const double* V, int32_t n_keys, int32_t Hkv, int32_t g,
                       int32_t D, double scale, double* x /* scratch [n_keys] */) {
    if (n_keys <= 0) {
        for (int32_t d = 0; d < D; ++d) out[d] = 0.0;
        if (lse) *lse = -INFINITY;
        return;
    }
    double M = -INFINITY;
    for (int32_t j = 0; j < n_keys; ++j) {
        const double* k = K + ((size_t)j * Hkv + g) * D;
        double acc = 0.0;
        for (int32_t d = 0; d < D; ++d) acc += bf16_to_f64(q_row[d]) * k[d];
        x[j] = scale * acc;
        if (x[j] > M) M = x[j];
    }
    double Z = 0.0;
    for (int32_t d = 0; d < D; ++d) out[d] = 0.0;
    for (int32_t j = 0; j < n_keys; ++j) {
        double w = exp(x[j] - M);
        x[j] = w;
        Z += w;
        const double* v = V + ((size_t)j * Hkv + g) * D;
        for (int32_t d = 0; d < D; ++d) out[d] += w * v[d];
    }
    for (int32_t d = 0; d < D; ++d) out[d] /= Z;
    if (lse) *lse = M + log(Z);
    if (probs)
        for (int32_t j = 0; j < n_keys; ++j) probs[j] = x[j] / Z;
}

/* DECODE.  out [S][Hq][D] fp64, lse [S][Hq] fp64 (may be NULL).  Returns 0, or -1 on bad geometry. */
int oracle_paged_decode(double* out, double* lse, const uint16_t* q, const uint16_t* k_pool,
                        const uint16_t* v_pool, const int32_t* block_table, int64_t block_table_stride,
                        const int32_t* seq_lens, int32_t S, int32_t Hq, int32_t Hkv, int32_t D,
                        int32_t p, double scale) {
    if (Hkv <= 0 || Hq % Hkv != 0) return -1;
    int32_t G = Hq / Hkv;
    for (int32_t s = 0; s < S; ++s) {
        int32_t L = seq_lens[s];
        size_t n = (size_t)(L > 0 ? L : 1) * Hkv * D;
        double* K = (double*)malloc(n * sizeof(double));
        double* V = (double*)malloc(n * sizeof(double));
        oracle_gather(K, V, k_pool, v_pool, block_table + (size_t)s * block_table_stride, L, Hkv, p, D);
#pragma omp parallel
        {
            double* x = (double*)malloc((size_t)(L > 0 ? L : 1) * sizeof(double));
#pragma omp for schedule(dynamic, 1)
            for (int32_t h = 0; h < Hq; ++h) {
                size_t r = (size_t)s * Hq + h;
                attend_row(out + r * D, lse ? lse + r : NULL, NULL, q + r * D, K, V, L, Hkv, h / G, D,
                           scale, x);
            }
            free(x);
        }
        free(K);
        free(V);
    }
    return 0;
}

/* P row of DECODE for one (s, h): probs [L_s] = w_j / Z.  Tiny inputs only (pin: rows sum to 1). */
int oracle_decode_probs(double* probs, const uint16_t* q, const uint16_t* k_pool, const uint16_t* v_pool,
                        const int32_t* block_table, int64_t block_table_stride, const int32_t* seq_lens,
                        int32_t s, int32_t h, int32_t Hq, int32_t Hkv, int32_t D, int32_t p, double scale) {
    if (Hkv <= 0 || Hq % Hkv != 0) return -1;
    int32_t L = seq_lens[s], G = Hq / Hkv;
    if (L <= 0) return 0;
    size_t n = (size_t)L * Hkv * D;
    double* K = (double*)malloc(n * sizeof(double));
    double* V = (double*)malloc(n * sizeof(double));
    double* x = (double*)malloc((size_t)L * sizeof(double));
    double* o = (double*)malloc((size_t)D * sizeof(double));
    oracle_gather(K, V, k_pool, v_pool, block_table + (size_t)s * block_table_stride, L, Hkv, p, D);
    attend_row(o, NULL, probs, q + ((size_t)s * Hq + h) * D, K, V, L, Hkv, h / G, D, scale, x);
    free(K); free(V); free(x); free(o);
    return 0;
}

/*
 * PREFILL over selected query rows.  rows [n_rows] are global row indices into q [T][Hq][D]
 * (ascending); out [n_rows][Hq][D], lse [n_rows][Hq] (may be NULL).  Sequence s owns rows
 * cu_seqlens_q[s] .. cu_seqlens_q[s+1]-1; local row i sees keys j <= P_s + i with
 * P_s = seq_lens[s] - n_s when causal != 0, else all L_s keys.
 */
int oracle_paged_prefill_rows(double* out, double* lse, const uint16_t* q, const int32_t* cu_seqlens_q,
                              const uint16_t* k_pool, const uint16_t* v_pool, const int32_t* block_table,
                              int64_t block_table_stride, const int32_t* seq_lens, int32_t S, int32_t Hq,
                              int32_t Hkv, int32_t D, int32_t p, double scale, int32_t causal,
                              const int32_t* rows, int64_t n_rows) {
    if (Hkv <= 0 || Hq % Hkv != 0) return -1;
    int32_t G = Hq / Hkv;
    int64_t a = 0;
    for (int32_t s = 0; s < S; ++s) {
        int32_t r0 = cu_seqlens_q[s], r1 = cu_seqlens_q[s + 1];
        int64_t b = a;
        while (b < n_rows && rows[b] < r1) ++b;
        if (b == a) continue; /* no selected row in this sequence */
        int32_t L = seq_lens[s], P = L - (r1 - r0);
        if (P < 0) return -2;
        size_t n = (size_t)(L > 0 ? L : 1) * Hkv * D;
        double* K = (double*)malloc(n * sizeof(double));
        double* V = (double*)malloc(n * sizeof(double));
        oracle_gather(K, V, k_pool, v_pool, block_table + (size_t)s * block_table_stride, L, Hkv, p, D);
        int64_t n_work = (b - a) * Hq;
#pragma omp parallel
        {
            double* x = (double*)malloc((size_t)(L > 0 ? L : 1) * sizeof(double));
#pragma omp for schedule(dynamic, 4)
            for (int64_t w = 0; w < n_work; ++w) {
                int64_t ri = a + w / Hq;
                int32_t h = (int32_t)(w % Hq);
                int32_t r = rows[ri];
                if (r < r0) continue; /* rows must be ascending; defensive */
                int32_t i = r - r0;
                int32_t n_keys = causal ? P + i + 1 : L;
                size_t o = (size_t)ri * Hq + h;
                attend_row(out + o * D, lse ? lse + o : NULL, NULL, q + ((size_t)r * Hq + h) * D, K, V,
                           n_keys, Hkv, h / G, D, scale, x);
            }
            free(x);
        }
        free(K);
        free(V);
        a = b;
    }
    return 0;
}

/*
 * One split-K partition of DECODE for (s, h): keys j0 <= j < j1 (clipped to L_s).
 * Writes m = max_j x_j, l = sum_j e^{x_j - m}, O[d] = sum_j e^{x_j - m} V[j][d] (UNnormalised).
 * Empty partition: m = -inf, l = 0, O = 0.
 */
int oracle_decode_partition(double* m_out, double* l_out, double* O, const uint16_t* q,
                            const uint16_t* k_pool, const uint16_t* v_pool, const int32_t* block_table,
                            int64_t block_table_stride, const int32_t* seq_lens, int32_t s, int32_t h,
                            int32_t Hq, int32_t Hkv, int32_t D, int32_t p, double scale, int32_t j0,
                            int32_t j1) {
    if (Hkv <= 0 || Hq % Hkv != 0) return -1;
    int32_t L = seq_lens[s], g = h / (Hq / Hkv);
    if (j1 > L) j1 = L;
    for (int32_t d = 0; d < D; ++d) O[d] = 0.0;
    *m_out = -INFINITY;
    *l_out = 0.0;
    if (j0 >= j1) return 0;
    size_t n = (size_t)L * Hkv * D;
    double* K = (double*)malloc(n * sizeof(double));
    double* V = (double*)malloc(n * sizeof(double));
    double* x = (double*)malloc((size_t)L * sizeof(double));
    oracle_gather(K, V, k_pool, v_pool, block_table + (size_t)s * block_table_stride, L, Hkv, p, D);
    const uint16_t* q_row = q + ((size_t)s * Hq + h) * D;
    double M = -INFINITY;
    for (int32_t j = j0; j < j1; ++j) {
        double acc = 0.0;
        for (int32_t d = 0; d < D; ++d) acc += bf16_to_f64(q_row[d]) * K[((size_t)j * Hkv + g) * D + d];
        x[j] = scale * acc;
        if (x[j] > M) M = x[j];
    }
    double l = 0.0;
    for (int32_t j = j0; j < j1; ++j) {
        double w = exp(x[j] - M);
        l += w;
        for (int32_t d = 0; d < D; ++d) O[d] += w * V[((size_t)j * Hkv + g) * D + d];
    }
    *m_out = M;
    *l_out = l;
    free(K); free(V); free(x);
    return 0;
}

/* COMBINE (step a3): merge n partitions of one row.  m, l [n]; O [n][D].  out [D], *lse. */
void oracle_lse_combine(double* out, double* lse, const double* m, const double* l, const double* O,
                        int32_t n, int32_t D) {
    double M = -INFINITY;
    for (int32_t i = 0; i < n; ++i)
        if (m[i] > M) M = m[i];
    for (int32_t d = 0; d < D; ++d) out[d] = 0.0;
    if (M == -INFINITY) { /* every partition empty: L = 0 */
        if (lse) *lse = -INFINITY;
        return;
    }
    double Z = 0.0;
    for (int32_t i = 0; i < n; ++i) {
        if (m[i] == -INFINITY) continue; /* e^{-inf} = 0 */
        double a = exp(m[i] - M);
        Z += a * l[i];
        for (int32_t d = 0; d < D; ++d) out[d] += a * O[(size_t)i * D + d];
    }
    for (int32_t d = 0; d < D; ++d) out[d] /= Z;
    if (lse) *lse = M + log(Z);
}


/* GATHER: pool -> contiguous [total][Hkv][D], 16-bit words. */
void oracle_kv_gather(uint16_t* k_out, uint16_t* v_out, const uint16_t* k_pool, const uint16_t* v_pool,
                      const int32_t* block_table, int64_t bt_stride, const int32_t* seq_lens,
                      const int32_t* cu_out, int32_t S, int32_t Hkv, int32_t p, int32_t D) {
    for (int32_t s = 0; s < S; ++s) {
        for (int32_t j = 0; j < seq_lens[s]; ++j) {
            int64_t page = block_table[(int64_t)s * bt_stride + j / p];
            int32_t off = j % p;
            for (int32_t h = 0; h < Hkv; ++h) {
                size_t src = (((size_t)page * Hkv + h) * p + off) * D;
                size_t dst = (((size_t)cu_out[s] + j) * Hkv + h) * D;
                for (int32_t d = 0; d < D; ++d) {
                    k_out[dst + d] = k_pool[src + d];
                    v_out[dst + d] = v_pool[src + d];
                }
            }
        }
    }
}

/* COPY_PAGES: whole pages between two pools of the same geometry (may be the same pool), sequential in i. */
void oracle_kv_copy_pages(uint16_t* k_dst, uint16_t* v_dst, const uint16_t* k_src, const uint16_t* v_src,
                          const int64_t* dst_pages, const int64_t* src_pages, int64_t n, int32_t Hkv, int32_t p,
                          int32_t D) {
    size_t page_elems = (size_t)Hkv * p * D;
    for (int64_t i = 0; i < n; ++i) {
        if (dst_pages[i] < 0 || src_pages[i] < 0) continue;
        for (size_t e = 0; e < page_elems; ++e) {
            k_dst[(size_t)dst_pages[i] * page_elems + e] = k_src[(size_t)src_pages[i] * page_elems + e];
            v_dst[(size_t)dst_pages[i] * page_elems + e] = v_src[(size_t)src_pages[i] * page_elems + e];
        }
    }
}
