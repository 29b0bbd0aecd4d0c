/*
 * oracle/attention_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct fp64 CPU definition of the mixed-batch paged
 * causal attention step that libcp (the CUDA path) computes.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may build, load or call this file.  It shares no code, header, table or
 * helper with paper_2606_09061_b200/csrc/.
 *
 * What it follows.  PAPER.md is silent on how attention is computed (the
 * execution backend is "unmodified"); the operation is the
 * textbook causal softmax attention over a paged KV cache (PAPER.md:41 cites
 * vLLM paged attention as the data structure; PAPER.md:61, :87 give the shape
 * of a chunked-prefill mixed batch).  The definition written out here is
 * SURVEY.md section 8(c1), restated:
 *
 *   for request j, row i in [0, q_len_j), q head h, g = h / G (G = Hq / Hkv),
 *   n = ctx_off_j + i + 1 keys are visible (diagonal inclusive):
 *     k_t = K[page = bt_j[t / B], slot = t % B, kv head g, :]   (same for v_t)
 *     s_t = sm_scale * sum_d q[tok(j,i), h, d] * k_t[d]             (fp64)
 *     m   = max_t s_t ;  p_t = exp(s_t - m)
 *     out[tok(j,i), h, :] = sum_t p_t v_t / sum_t p_t     (two-pass softmax)
 *
 * No blocking, no online softmax, no fusion: one (row, head) at a time.
 *
 * Cache layout (the ABI of include/cp.h, indexed here independently):
 *   kv_cache[block][kv (0 = K, 1 = V)][kv_head][slot][d]   bf16, one layer.
 *
 * Inputs are bf16 BIT PATTERNS (uint16) widened exactly to fp64.
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 *
 * Pins (tests/test_oracle_attention.py): brute-force dense L x L softmax,
 * torch SDPA fp64, chunking invariance, decode consistency, closed forms,
 * block-table permutation / GQA replication / poison invariants.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static inline double bf16_to_f64(uint16_t b)
{
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* element offset of (block, kv, head, slot, 0) in the single-layer pool */
static inline int64_t cache_row(int64_t block, int kv, int head, int slot,
                                int Hkv, int B, int D)
{
    return ((((int64_t)block * 2 + kv) * Hkv + head) * B + slot) * (int64_t)D;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * KV append: the iteration's new K,V rows go to their pages
 * before anything attends.  Token i of request j has absolute position
 * p = ctx_off_j + i -> page bt_j[p / B], slot p % B.
 * k_new, v_new: [T, Hkv, D] bf16 bits, token order = descriptor order.
 * bt_off[j] .. bt_off[j+1] delimit request j's page ids in block_table.
 * Returns 0, or -1 if a request's table is too short / page id out of range.
 */
int oracle_kv_append(const uint16_t *k_new, const uint16_t *v_new,
                     uint16_t *kv_cache, const int32_t *q_len,
                     const int32_t *ctx_off, const int32_t *bt_off,
                     const int32_t *block_table, int n_reqs, int Hkv, int D,
                     int B, int64_t num_blocks)
{
    int64_t tok = 0;
    for (int j = 0; j < n_reqs; ++j) {
        const int32_t *bt = block_table + bt_off[j];
        int nb = bt_off[j + 1] - bt_off[j];
        for (int i = 0; i < q_len[j]; ++i, ++tok) {
            int64_t p = (int64_t)ctx_off[j] + i;
            if (p / B >= nb) return -1;
            int64_t page = bt[p / B];
            if (page < 0 || page >= num_blocks) return -1;
            int slot = (int)(p % B);
            for (int g = 0; g < Hkv; ++g) {
                const uint16_t *ks = k_new + (tok * Hkv + g) * D;
                const uint16_t *vs = v_new + (tok * Hkv + g) * D;
                memcpy(kv_cache + cache_row(page, 0, g, slot, Hkv, B, D), ks,
                       sizeof(uint16_t) * D);
                memcpy(kv_cache + cache_row(page, 1, g, slot, Hkv, B, D), vs,
                       sizeof(uint16_t) * D);
            }
        }
    }
    return 0;
}

/*
 * Attention for a list of (token, head) rows.
 *   q          [T, Hq, D] bf16 bits
 *   kv_cache   single-layer pool, already holding this iteration's K/V
 *   q_len, ctx_off [n_reqs]; bt_off [n_reqs+1]; block_table flat page ids
 *   row_tok[r], row_head[r] for r in [0, n_rows): global token index (in
 *   descriptor order) and q head of the r-th row to compute.  Passing
 *   row_tok == NULL means "all T*Hq rows in (token, head) order".
 *   out        [n_rows, D] fp64
 * Returns 0 on success, -1 on bad arguments.
 */
int oracle_attention_rows(const uint16_t *q, const uint16_t *kv_cache,
                          const int32_t *q_len, const int32_t *ctx_off,
                          const int32_t *bt_off, const int32_t *block_table,
                          int n_reqs, int Hq, int Hkv, int D, int B,
                          int64_t num_blocks, double sm_scale,
                          const int64_t *row_tok, const int32_t *row_head,
                          int64_t n_rows, double *out)
{
    if (Hkv <= 0 || Hq % Hkv != 0 || D <= 0 || B <= 0) return -1;
    const int G = Hq / Hkv;

    /* token -> (request, row-in-request) map */
    int64_t T = 0;
    for (int j = 0; j < n_reqs; ++j) T += q_len[j];
    int32_t *tok_req = (int32_t *)malloc(sizeof(int32_t) * (size_t)(T > 0 ? T : 1));
    int32_t *tok_row = (int32_t *)malloc(sizeof(int32_t) * (size_t)(T > 0 ? T : 1));
    if (!tok_req || !tok_row) { free(tok_req); free(tok_row); return -1; }
    {
        int64_t t = 0;
        for (int j = 0; j < n_reqs; ++j)
            for (int i = 0; i < q_len[j]; ++i, ++t) { tok_req[t] = j; tok_row[t] = i; }
    }
    if (row_tok == NULL) n_rows = T * Hq;

    int bad = 0;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t r = 0; r < n_rows; ++r) {
        int64_t tok = row_tok ? row_tok[r] : r / Hq;
        int h = row_tok ? row_head[r] : (int)(r % Hq);
        if (tok < 0 || tok >= T || h < 0 || h >= Hq) { bad = 1; continue; }
        int j = tok_req[tok];
        int i = tok_row[tok];
        int g = h / G;                         /* consecutive GQA grouping */
        int64_t n = (int64_t)ctx_off[j] + i + 1; /* visible keys, diagonal incl. */
        const int32_t *bt = block_table + bt_off[j];
        int nb = bt_off[j + 1] - bt_off[j];
        if ((n + B - 1) / B > nb) { bad = 1; continue; }

        double *qd = (double *)malloc(sizeof(double) * (size_t)D);
        double *s = (double *)malloc(sizeof(double) * (size_t)n);
        double *o = out + r * (int64_t)D;
        for (int d = 0; d < D; ++d) qd[d] = bf16_to_f64(q[(tok * Hq + h) * D + d]);

        /* pass 1: scores and their max */
        double m = -INFINITY;
        for (int64_t t = 0; t < n; ++t) {
            int64_t page = bt[t / B];
            if (page < 0 || page >= num_blocks) { bad = 1; page = 0; }
            const uint16_t *kr =
                kv_cache + cache_row(page, 0, g, (int)(t % B), Hkv, B, D);
            double acc = 0.0;
            for (int d = 0; d < D; ++d) acc += qd[d] * bf16_to_f64(kr[d]);
            s[t] = sm_scale * acc;
            if (s[t] > m) m = s[t];
        }
        /* pass 2: weights, weighted sum of V, normalise */
        double l = 0.0;
        for (int d = 0; d < D; ++d) o[d] = 0.0;
        for (int64_t t = 0; t < n; ++t) {
            int64_t page = bt[t / B];
            if (page < 0 || page >= num_blocks) page = 0;
            const uint16_t *vr =
                kv_cache + cache_row(page, 1, g, (int)(t % B), Hkv, B, D);
            double p = exp(s[t] - m);
            l += p;
            for (int d = 0; d < D; ++d) o[d] += p * bf16_to_f64(vr[d]);
        }
        for (int d = 0; d < D; ++d) o[d] /= l;
        free(qd);
        free(s);
    }
    free(tok_req);
    free(tok_row);
    return bad ? -1 : 0;
}
