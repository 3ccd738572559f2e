/*
 * tropical_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU fp64 definition of what one multiplexed worker
 * iteration computes (PAPER.md:143, :159 -- a prefill chunk co-run with the decode batch of
 * one worker; the paper inherits the attention itself from its vLLM/PagedAttention substrate,
 * PAPER.md:182, :224, :246).  BASELINE.json north_star fixes the definition:
 * "softmax(QK^T/sqrt(d) + causal mask)V over gathered pages", fp64, after the KV append.
 * SURVEY.md section 8(c) restates it with the readings S1-S28; DESIGN.md lists them.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code with paper_2606_16264_b200/.
 *
 * The GPU path reaches exactly this result by re-association (tiling, online softmax,
 * split-K, paging), so the oracle is the definition written out -- no blocking, no fusion,
 * no online softmax.  Every score of a row is materialised, then max, then sum, then the
 * weighted sum over values.
 *
 * Pins (tests/test_oracle_pins.py): brute-force dense attention, torch fp64 SDPA, closed
 * forms, row-sum-to-one, page-size and page-permutation invariance, chunk/decode
 * consistency, needle selection; kv_migrate: gather(dst) == gather(src) by fancy indexing, changed-row
 * count, attention unchanged by the move; RoPE append: identity table == plain append, quarter-turn table == swap
 * and negate, norm and relative-position invariants, position indexing, rounding against ties worked by hand.
 * Step-cost model: not in this file (parity unpinned).
 *
 * Layouts (host pointers, bf16 carried as uint16 bit patterns):
 *   q            [T][Hq][d]           k_new, v_new [T][Hkv][d]
 *   k_pool/v_pool [num_pages][Hkv][P][d]
 *   page_table   [num_reqs][stride]   q_lens, ctx_lens [num_reqs]   q_offsets [num_reqs+1]
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

static inline double bf16_to_double(uint16_t b)
{
    uint32_t u = ((uint32_t)b) << 16; /* bf16 is the top half of an IEEE binary32 */
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Phase 1 -- KV append (reading S4 "append-all then attend").
 * for t < q_i: pos = c_i + t; page = page_table[i][pos / P]; slot = pos % P;
 * pool[page][h][slot][:] = new[q_off_i + t][h][:]   -- raw 16-bit copies, no FP. */
void oracle_kv_append(int Hkv, int d, int P, int num_reqs, const int32_t *q_lens,
                      const int32_t *ctx_lens, const int32_t *q_offsets,
                      const int32_t *page_table, int stride, uint16_t *k_pool, uint16_t *v_pool,
                      const uint16_t *k_new, const uint16_t *v_new)
{
    for (int i = 0; i < num_reqs; ++i) {
        for (int t = 0; t < q_lens[i]; ++t) {
            int64_t pos = (int64_t)ctx_lens[i] + t;
            int64_t page = page_table[(int64_t)i * stride + pos / P];
            int64_t slot = pos % P;
            for (int h = 0; h < Hkv; ++h) {
                int64_t dst = ((page * Hkv + h) * P + slot) * d;
                int64_t src = (((int64_t)q_offsets[i] + t) * Hkv + h) * d;
                for (int c = 0; c < d; ++c) {
                    k_pool[dst + c] = k_new[src + c];
                    v_pool[dst + c] = v_new[src + c];
                }
            }
        }
    }
}

/* Page gather (row A2): logical key j of request i -> (page_table[i][j / P], j % P).
 * Dense copy-out of the first n_keys keys of request req: k_dense/v_dense [n_keys][Hkv][d]. */
void oracle_kv_gather(int Hkv, int d, int P, const int32_t *page_table, int stride, int req,
                      int n_keys, const uint16_t *k_pool, const uint16_t *v_pool,
                      uint16_t *k_dense, uint16_t *v_dense)
{
    for (int j = 0; j < n_keys; ++j) {
        int64_t page = page_table[(int64_t)req * stride + j / P];
        int64_t slot = j % P;
        for (int h = 0; h < Hkv; ++h) {
            int64_t src = ((page * Hkv + h) * P + slot) * d;
            int64_t dst = ((int64_t)j * Hkv + h) * d;
            for (int c = 0; c < d; ++c) {
                k_dense[dst + c] = k_pool[src + c];
                v_dense[dst + c] = v_pool[src + c];
            }
        }
    }
}

/* KV migration (PAPER.md:155 Path 1: after its prefill on a prefill worker a request
 * re-enters through the decode queue and its KV cache moves to the multiplexing worker that will decode it;
 * PAPER.md:58, :101 "migration of KVCache"; :171 P2P between GPUs).  The paper fixes nothing below "the cache
 * moves"; the reading is token-granular and page-table to page-table:
 *   for request m, j < kv_lens[m], h < Hkv:
 *     dst_pool[dst_pt[m][j / P]][h][j % P][:] = src_pool[src_pt[m][j / P]][h][j % P][:]      (K and V)
 * Raw 16-bit copies.  Slots j >= kv_lens[m] of a destination page and every other destination page keep
 * their bits; the source pools are read-only. */
void oracle_kv_migrate(int Hkv, int d, int P, int num_reqs, const int32_t *kv_lens,
                       const int32_t *src_pt, int src_stride, const int32_t *dst_pt, int dst_stride,
                       const uint16_t *k_src, const uint16_t *v_src, uint16_t *k_dst, uint16_t *v_dst)
{
    for (int m = 0; m < num_reqs; ++m) {
        for (int64_t j = 0; j < kv_lens[m]; ++j) {
            int64_t sp = src_pt[(int64_t)m * src_stride + j / P];
            int64_t dp = dst_pt[(int64_t)m * dst_stride + j / P];
            int64_t slot = j % P;
            for (int h = 0; h < Hkv; ++h) {
                int64_t so = ((sp * Hkv + h) * P + slot) * d;
                int64_t dof = ((dp * Hkv + h) * P + slot) * d;
                for (int c = 0; c < d; ++c) {
                    k_dst[dof + c] = k_src[so + c];
                    v_dst[dof + c] = v_src[so + c];
                }
            }
        }
    }
}

/* SURVEY 8(f) NEXT-4 "fuse RoPE+append": rotary position embedding of this step's K rows on their way into the pool.
 * The paper says nothing about positional encoding (its substrate's models use it); the definition taken
 * is the "rotate-half" convention of that model family [DESIGN.md reading R-rope]: channel c < d/2 is paired with
 * channel c + d/2, the token at position pos = c_i + t uses row pos of the caller's tables cos, sin [table_len][d/2]:
 *     k'[c]       = k[c] * cos[pos][c] - k[c + d/2] * sin[pos][c]
 *     k'[c + d/2] = k[c + d/2] * cos[pos][c] + k[c] * sin[pos][c]
 * The products of a bf16 value (8 significant bits) and an fp32 value (24) are exact in fp64 and so is their sum
 * unless the exponents are far apart, so out[] below is the real-number result to fp64 accuracy. */
void oracle_rope_rotate(int d, int64_t n_rows, const uint16_t *rows, const int32_t *pos, const float *cos_t,
                        const float *sin_t, double *out)
{
    const int half = d / 2;
    for (int64_t r = 0; r < n_rows; ++r) {
        for (int c = 0; c < half; ++c) {
            double x = bf16_to_double(rows[r * d + c]), y = bf16_to_double(rows[r * d + c + half]);
            double cs = (double)cos_t[(int64_t)pos[r] * half + c], sn = (double)sin_t[(int64_t)pos[r] * half + c];
            out[r * d + c] = x * cs - y * sn;
            out[r * d + c + half] = y * cs + x * sn;
        }
    }
}

/* fp64 -> bf16, round to nearest even, straight from the double (no intermediate fp32 rounding).  Finite inputs
 * within the bf16 normal range, +-0 and values that round to +-0 / subnormals are flushed by magnitude < 2^-126 -> 0
 * (the rotated N(0,1) data of the tests never get there); NaN / inf pass through as the bf16 patterns. */
uint16_t oracle_double_to_bf16(double v)
{
    uint64_t u;
    memcpy(&u, &v, sizeof u);
    uint16_t sign = (uint16_t)((u >> 63) << 15);
    int64_t e = (int64_t)((u >> 52) & 0x7ff);
    uint64_t m = u & 0xfffffffffffffULL;
    if (e == 0x7ff) return (uint16_t)(sign | 0x7f80 | (m ? 0x40 : 0));
    int64_t eb = e - 1023 + 127;                  /* bf16 / fp32 biased exponent */
    if (e == 0 || eb <= 0) return sign;           /* zero, fp64 subnormal, or below the bf16 normal range */
    uint64_t keep = m >> 45;                      /* top 7 mantissa bits */
    uint64_t rest = m & ((1ULL << 45) - 1), half = 1ULL << 44;
    if (rest > half || (rest == half && (keep & 1))) ++keep;
    if (keep == 128) { keep = 0; ++eb; }
    if (eb >= 255) return (uint16_t)(sign | 0x7f80);
    return (uint16_t)(sign | (uint16_t)(eb << 7) | (uint16_t)keep);
}

/* Append with RoPE on K: the row that oracle_kv_append would copy is rotated (oracle_rope_rotate), rounded to bf16
 * (oracle_double_to_bf16) and stored; V rows are copied.  Row by row, in the paper-free definition's order. */
void oracle_kv_append_rope(int Hkv, int d, int P, int num_reqs, const int32_t *q_lens,
                           const int32_t *ctx_lens, const int32_t *q_offsets,
                           const int32_t *page_table, int stride, uint16_t *k_pool, uint16_t *v_pool,
                           const uint16_t *k_new, const uint16_t *v_new, const float *cos_t, const float *sin_t)
{
    double *rot = (double *)malloc(sizeof(double) * (size_t)d);
    for (int i = 0; i < num_reqs; ++i) {
        for (int t = 0; t < q_lens[i]; ++t) {
            int64_t pos = (int64_t)ctx_lens[i] + t;
            int32_t pos32 = (int32_t)pos;
            int64_t page = page_table[(int64_t)i * stride + pos / P];
            int64_t slot = pos % P;
            for (int h = 0; h < Hkv; ++h) {
                int64_t dst = ((page * Hkv + h) * P + slot) * d;
                int64_t src = (((int64_t)q_offsets[i] + t) * Hkv + h) * d;
                oracle_rope_rotate(d, 1, k_new + src, &pos32, cos_t, sin_t, rot);
                for (int c = 0; c < d; ++c) {
                    k_pool[dst + c] = oracle_double_to_bf16(rot[c]);
                    v_pool[dst + c] = v_new[src + c];
                }
            }
        }
    }
    free(rot);
}

/* One (request i, new-token t, q-head hq) row of phase 2 (rows A3/A4/A5 all compute this):
 *   hk = hq / (Hq/Hkv)                        (S6: contiguous GQA groups)
 *   n  = c_i + t + 1                          (S3: causal, bottom-right aligned; S4: sees itself)
 *   s_j = scale * sum_c q[c] * K_j[c]         j in [0, n)
 *   m = max_j s_j;  Z = sum_j exp(s_j - m);   w_j = exp(s_j - m) / Z
 *   out[c] = sum_j w_j * V_j[c];              lse = m + log Z;   wsum = sum_j w_j
 * scratch s: n doubles. */
static void attention_row(int Hq, int Hkv, int d, int P, const int32_t *ctx_lens,
                          const int32_t *q_offsets, const int32_t *page_table, int stride,
                          const uint16_t *k_pool, const uint16_t *v_pool, const uint16_t *q,
                          double scale, int i, int t, int hq, double *s, double *out, double *lse,
                          double *wsum)
{
    const int g = Hq / Hkv;
    const int hk = hq / g;
    const int64_t n = (int64_t)ctx_lens[i] + t + 1;
    const uint16_t *qrow = q + (((int64_t)q_offsets[i] + t) * Hq + hq) * d;
    const int32_t *pt = page_table + (int64_t)i * stride;

    for (int64_t j = 0; j < n; ++j) {
        const uint16_t *krow = k_pool + (((int64_t)pt[j / P] * Hkv + hk) * P + j % P) * d;
        double acc = 0.0;
        for (int c = 0; c < d; ++c) acc += bf16_to_double(qrow[c]) * bf16_to_double(krow[c]);
        s[j] = scale * acc;
    }
    double m = s[0];
    for (int64_t j = 1; j < n; ++j) m = s[j] > m ? s[j] : m;
    double Z = 0.0;
    for (int64_t j = 0; j < n; ++j) Z += exp(s[j] - m);
    for (int c = 0; c < d; ++c) out[c] = 0.0;
    double ws = 0.0;
    for (int64_t j = 0; j < n; ++j) {
        const uint16_t *vrow = v_pool + (((int64_t)pt[j / P] * Hkv + hk) * P + j % P) * d;
        double w = exp(s[j] - m) / Z;
        ws += w;
        for (int c = 0; c < d; ++c) out[c] += w * bf16_to_double(vrow[c]);
    }
    if (lse) *lse = m + log(Z);
    if (wsum) *wsum = ws;
}

/* Phase 2 on a chosen subset of rows: row r is (row_req[r], row_t[r]) with 0 <= t < q_lens[req].
 * out [n_rows][Hq][d], lse (nullable) [n_rows][Hq], wsum (nullable) [n_rows][Hq].
 * scale <= 0 selects 1/sqrt(d) (S2).  Returns 0, or -1 if scratch allocation failed. */
int oracle_attention_rows(int Hq, int Hkv, int d, int P, const int32_t *q_lens,
                          const int32_t *ctx_lens, const int32_t *q_offsets,
                          const int32_t *page_table, int stride, const uint16_t *k_pool,
                          const uint16_t *v_pool, const uint16_t *q, double scale, int n_rows,
                          const int32_t *row_req, const int32_t *row_t, double *out, double *lse,
                          double *wsum)
{
    (void)q_lens;
    if (!(scale > 0.0)) scale = 1.0 / sqrt((double)d);
    int64_t max_n = 1;
    for (int r = 0; r < n_rows; ++r) {
        int64_t n = (int64_t)ctx_lens[row_req[r]] + row_t[r] + 1;
        if (n > max_n) max_n = n;
    }
    int failed = 0;
#pragma omp parallel
    {
        double *s = (double *)malloc(sizeof(double) * (size_t)max_n);
        if (!s) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp for collapse(2) schedule(dynamic, 4)
        for (int r = 0; r < n_rows; ++r) {
            for (int hq = 0; hq < Hq; ++hq) {
                if (!s) continue;
                int64_t o = (int64_t)r * Hq + hq;
                attention_row(Hq, Hkv, d, P, ctx_lens, q_offsets, page_table, stride, k_pool,
                              v_pool, q, scale, row_req[r], row_t[r], hq, s, out + o * d,
                              lse ? lse + o : 0, wsum ? wsum + o : 0);
            }
        }
        free(s);
    }
    return failed ? -1 : 0;
}

/* Phase 2 on every row of the step: out [T][Hq][d], lse/wsum (nullable) [T][Hq]. */
int oracle_mixed_attention(int Hq, int Hkv, int d, int P, int num_reqs, const int32_t *q_lens,
                           const int32_t *ctx_lens, const int32_t *q_offsets,
                           const int32_t *page_table, int stride, const uint16_t *k_pool,
                           const uint16_t *v_pool, const uint16_t *q, double scale, double *out,
                           double *lse, double *wsum)
{
    int64_t T = q_offsets[num_reqs];
    if (T == 0) return 0;
    int32_t *row_req = (int32_t *)malloc(sizeof(int32_t) * (size_t)T);
    int32_t *row_t = (int32_t *)malloc(sizeof(int32_t) * (size_t)T);
    if (!row_req || !row_t) {
        free(row_req);
        free(row_t);
        return -1;
    }
    for (int i = 0; i < num_reqs; ++i)
        for (int t = 0; t < q_lens[i]; ++t) {
            row_req[q_offsets[i] + t] = i;
            row_t[q_offsets[i] + t] = t;
        }
    int rc = oracle_attention_rows(Hq, Hkv, d, P, q_lens, ctx_lens, q_offsets, page_table, stride,
                                   k_pool, v_pool, q, scale, (int)T, row_req, row_t, out, lse, wsum);
    free(row_req);
    free(row_t);
    return rc;
}
