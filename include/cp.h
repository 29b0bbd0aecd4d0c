/*
 * cp.h -- C ABI of libcp: the mixed-batch paged-attention step of a chunked-prefill
 * serving iteration on one NVIDIA B200 (sm_100a), plus the host-side scheduler that
 * forms each iteration (aging / LPRS / APC of arxiv/paper_2606_09061).
 *
 * Plain C, plain pointers, no torch types.  Every pointer argument says whether it is
 * HOST or DEVICE memory.  All functions return int: CP_OK (0) or a negative error;
 * nothing throws or aborts; cp_last_error() gives a thread-local message.
 *
 * Ownership: the caller owns every device tensor it passes (q, k_new, v_new, kv_cache,
 * out) and the CUDA stream.  The library owns its context, device metadata, the
 * split-KV partial workspace, pinned staging, a copy stream and CUDA events, all
 * allocated in cp_create from the limits in cp_config; nothing is allocated afterwards.
 * Calls that may block the host: cp_latency_table (waits for the newest timed step),
 * cp_destroy, cp_enable_rope, and cp_build_batch ONLY when the host runs more than three
 * batches ahead of the device (the metadata staging ring is four batches deep).
 *
 * The operation (PAPER.md:61, :87 chunked-prefill mixed batch; PAPER.md:41 paged KV;
 * defined in DESIGN.md section 2, restating SURVEY.md 8(c1)): for request j, row
 * i < q_len_j, q head h, g = h / (Hq/Hkv), over keys t in [0, ctx_off_j + i]:
 *     s_t = sm_scale * <q[tok(j,i),h,:], K_j[t,g,:]>,  out = softmax_t(s) . V_j[:,g,:]
 * where K_j[t], V_j[t] live in page block_table_j[t / B], slot t % B.  A decode is
 * simply q_len == 1.  Stale data in page tails / other pages never influences the
 * result, whatever its bit pattern (NaN and Inf included): masked scores are removed by
 * select, and every step first ZEROES the slots of each request's last page that lie past
 * its last key (they belong to the request, hold no key, and later appends overwrite
 * them), so that masked P = 0 never meets a NaN in the tensor-core PV product.
 */
#ifndef CP_H_
#define CP_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CP_OK          0
#define CP_EINVAL     (-1)   /* bad argument / shape / table too short            */
#define CP_ECAPACITY  (-2)   /* exceeds a limit fixed at cp_create               */
#define CP_ECUDA      (-3)   /* a CUDA call failed (message in cp_last_error)     */
#define CP_ESTATE     (-4)   /* wrong call order (e.g. step before build_batch)   */

#define CP_NUM_RAW_FEATURES 11   /* Table 1 */
#define CP_NUM_FEATURES     16   /* + Table 2 */

typedef struct cp_ctx cp_ctx;       /* opaque */
typedef struct cp_sched cp_sched;   /* opaque */

/* ---------------------------------------------------------------------------------
 * KV cache layout (part of the ABI), bf16, one pool per layer, layer-major:
 *     kv_cache[layer][block][kv: 0 = K, 1 = V][kv_head][slot in 0..B-1][d in 0..D-1]
 * A (block, kv, head) slab is B*D*2 bytes contiguous (4 KiB at B 16, D 128); K and V
 * of a block are adjacent.  cp_attention_step takes the pointer to the LAYER's pool.
 * The pool needs no initialisation (a torch.empty pool is fine).
 * ------------------------------------------------------------------------------- */
typedef struct {
    int32_t num_q_heads;      /* Hq                                               */
    int32_t num_kv_heads;     /* Hkv, divides Hq; G = Hq/Hkv in {1,2,4,8,16}      */
    int32_t head_dim;         /* D in {64, 128}                                   */
    int32_t block_size;       /* B, tokens per page: 16                           */
    int32_t num_layers;       /* only used to size the latency ring; >= 1         */
    int64_t num_blocks;       /* pages per layer pool                             */
    float   sm_scale;         /* e.g. 1/sqrt(D), applied in fp32                  */
    int32_t max_tokens;       /* limit on T = sum q_len per batch                 */
    int32_t max_reqs;         /* limit on requests per batch                      */
    int64_t max_total_pages;  /* limit on sum of n_blocks over the batch          */
    int64_t max_partial_rows; /* split-KV workspace rows ((D+2) fp32 each);
                                 0 = default 4 * max_tokens * Hq                  */
    int32_t device;           /* CUDA device ordinal                              */
    int32_t kernel_variant;   /* must be 0.  (Library builds with -DCP_DEBUG_VARIANTS also
                                 accept 1 = a SIMT cross-check kernel for bisecting; the
                                 shipped library holds one attention kernel and rejects it.) */
    int32_t kv_dtype;         /* CP_KV_BF16 (0) or CP_KV_E4M3 (1): format of the KV pool.  E4M3
                                 pools are driven through cp_attention_step_fp8 (D = 128 only) */
    int32_t reserved;         /* must be 0                                          */
    int64_t max_scratch_pages;/* CP_KV_E4M3 only: pages of the library's bf16 scratch pool that
                                 holds, per step, the dequantised pages of the requests with a
                                 prefill chunk (> 8 rows per KV head); 0 = max_total_pages */
} cp_config;
#define CP_KV_BF16 0
#define CP_KV_E4M3 1

/* One request of the iteration.  HOST pointers. */
#define CP_REQ_PREFILL 1         /* flags: this request is in its prefill phase   */
typedef struct {
    int64_t        req_id;
    int32_t        q_len;        /* >= 1 tokens scheduled this iteration          */
    int32_t        ctx_off;      /* >= 0 tokens already in the cache before them  */
    const int32_t* block_table;  /* HOST: n_blocks page ids in [0, num_blocks)    */
    int32_t        n_blocks;     /* n_blocks * B >= ctx_off + q_len               */
    int32_t        flags;        /* CP_REQ_PREFILL or 0.  Only the Table-1 features and
                                    n_prefill / n_decode of cp_latency_row read it: a
                                    1-token prefill chunk (Eq. 8's candidate c = 1, the last
                                    token of a prompt) counts as prefill there, as in the
                                    scheduler's own features.  q_len > 1 is always prefill.
                                    The computation is the same either way.            */
} cp_req_desc;

/* One timed step: the 11 raw features of Table 1 + measured us
 * ("ground-truth batch latency measured by a high-resolution timer"). */
typedef struct {
    float   feat[CP_NUM_RAW_FEATURES]; /* prefill_tokens, decode_tokens,
          batch_request_count, sum_decode_context_len, max_decode_context_len,
          prefill_processed_tokens, max_prefill_processed_tokens, gpu_mem_used_mb,
          gpu_mem_free_mb, cuda_allocated_mb, cuda_reserved_mb                    */
    float   us;                 /* device time of cp_attention_step (CUDA events)  */
    int32_t n_prefill;          /* requests with q_len > 1 or CP_REQ_PREFILL       */
    int32_t n_decode;           /* the others                                      */
    int32_t layer;              /* >= 0: the layer of a cp_attention_step; -n: n layers timed together (cp_attention_layers) */
    int64_t iter;               /* index of the cp_build_batch this step ran under */
} cp_latency_row;

const char* cp_last_error(void);

/* Create / destroy a context.  cfg: HOST.  Allocates everything the context will ever
 * need.  Errors: CP_EINVAL (unsupported shape), CP_ECUDA. */
int cp_create(const cp_config* cfg, cp_ctx** out);
int cp_destroy(cp_ctx* ctx);

/* H1: pack the iteration's request descriptors into device metadata
 * (cu_q, q_len, ctx_off, flat block table, work list, combine list) with ONE async
 * host->device copy on `cuda_stream` (a cudaStream_t, may be NULL = default stream).
 * reqs: HOST array of n_reqs descriptors, any mix/order of prefill chunks and decodes;
 * token order of q/out = descriptor order, rows of a request contiguous.
 * A page id may appear in only one request of the batch (no prefix sharing); this is NOT
 * checked (a duplicate with k_new set is a write race) except in -DCP_DEBUG_VARIANTS
 * builds, which return CP_EINVAL.  The metadata stays valid for any number of
 * cp_attention_step calls (all layers) until the next cp_build_batch; its host->device
 * copy runs on the library's copy stream, overlapping the previous batch's steps, and
 * `cuda_stream` waits for it.  All steps of a batch must run on one stream (or on
 * streams the caller orders after it).
 * Errors: CP_EINVAL (q_len < 1, ctx_off < 0, table too short, page id out of range),
 * CP_ECAPACITY (limits of cp_config), CP_ECUDA.  On error the previous batch is kept. */
int cp_build_batch(cp_ctx* ctx, const cp_req_desc* reqs, int32_t n_reqs,
                   void* cuda_stream);

/* H2-H6: run the attention step of one layer for the current batch, asynchronously on
 * `cuda_stream`, bracketed by a CUDA-event pair that cp_latency_table later resolves.
 *   q        DEVICE [T, Hq, D]  bf16
 *   k_new    DEVICE [T, Hkv, D] bf16, or NULL = caller already wrote the pages
 *   v_new    DEVICE [T, Hkv, D] bf16 (NULL iff k_new is NULL)
 *   kv_cache DEVICE the layer's pool [num_blocks][2][Hkv][B][D] bf16; the new rows are
 *            appended in place before anything attends (H2); the unused slots of each
 *            request's last page are zeroed (also when k_new is NULL); nothing else is written
 *   out      DEVICE [T, Hq, D]  bf16, every row written
 * All pointers 16-byte aligned.  Errors: CP_ESTATE (no batch built), CP_EINVAL, CP_ECUDA. */
int cp_attention_step(cp_ctx* ctx, int32_t layer, const void* q, const void* k_new,
                      const void* v_new, void* kv_cache, void* out, void* cuda_stream);

/* All layers of the iteration in ONE submission (PAPER.md:201 names kernel launch latency among the fixed
 * per-round overheads; most rounds of a serving trace are a handful of decodes, where the per-call cost is the
 * bulk of the time): exactly the kernels of n_layers cp_attention_step calls with layer = 0 .. n_layers-1, but
 * one host call, ONE CUDA-event pair and one cp_latency_row for the whole iteration (its `layer` is -n_layers,
 * its `us` the time of all layers).  q, k_new, v_new, kv_cache, out: HOST arrays of n_layers DEVICE pointers
 * (k_new and v_new may both be NULL).  bf16 pools only.  Errors as cp_attention_step. */
int cp_attention_layers(cp_ctx* ctx, int32_t n_layers, const void* const* q, const void* const* k_new,
                        const void* const* v_new, void* const* kv_cache, void* const* out, void* cuda_stream);

/* N2 of SURVEY.md 8(f): rotary position embedding fused into the append (H2).  PAPER.md is
 * silent on positional encoding (the execution backend is untouched); the
 * definition is the textbook rotary embedding in the rotate-half pairing (R11): a row
 * x of D elements at absolute position p = ctx_off + i becomes, for f in [0, D/2),
 *     x'[f]       = x[f] cos(p w_f) - x[f + D/2] sin(p w_f)
 *     x'[f + D/2] = x[f + D/2] cos(p w_f) + x[f] sin(p w_f)
 * Angles and their cos / sin are evaluated in fp64 and rounded to fp32; products and sums are
 * fp32 without fused multiply-add; the result is rounded to nearest even bf16 (R12).
 *
 * cp_enable_rope: inv_freq HOST [D/2] finite doubles (w_f; the usual choice is theta^(-2f/D)),
 * copied.  A set-up call: allocates the rotated-Q workspace [max_tokens, Hq, D] bf16 and the
 * (cos, sin) table [max_tokens, D/2], synchronises the device; may be called again to change the
 * frequencies.  Batches built afterwards carry their table (one small kernel per cp_build_batch).
 * Errors: CP_EINVAL, CP_ECUDA.
 *
 * cp_attention_step_rope: as cp_attention_step, but q and k_new are UNROTATED: K rows are rotated
 * on their way into the pages, Q rows into the library's workspace (q itself is not modified), V
 * rows are copied, all in the one append kernel; everything then attends as in cp_attention_step.
 * k_new / v_new must not be NULL.  Errors: CP_ESTATE (cp_enable_rope not called, or the current
 * batch was built before it), CP_EINVAL, CP_ECUDA. */
int cp_enable_rope(cp_ctx* ctx, const double* inv_freq);
int cp_attention_step_rope(cp_ctx* ctx, int32_t layer, const void* q, const void* k_new,
                           const void* v_new, void* kv_cache, void* out, void* cuda_stream);

/* N2 of SURVEY.md 8(f), second half: FP8 (e4m3) KV pages -- half the bytes of the memory-bound decode
 * streams ("decode ... memory-bandwidth-bound").  PAPER.md defines none of it; DESIGN.md
 * R13-R15.  Pool layout (ABI), one pool per layer:
 *     kv_cache8[block][kv: 0 = K, 1 = V][kv_head][slot 0..B-1][d 0..D-1]   uint8, OCP FP8 E4M3 codes
 *     kv_scale [block][kv][kv_head][slot]                                  float32, a power of two 2^e
 * The value a slot holds is code_value * 2^e exactly.  Appended rows are quantised row by row: e = the smallest
 * integer with 448 * 2^e >= amax(row), clamped to [-15, 7]; code = round-to-nearest-even of x * 2^-e, saturating
 * at +-448 (oracle/kv_fp8.py is the definition the tests hold the library to, bit for bit).  Attention is the
 * operation above over those values; the output tolerance is the same.
 *   q, k_new, v_new  DEVICE bf16 as in cp_attention_step (k_new / v_new may be NULL: the caller wrote codes
 *                    and scales itself); kv_cache8 DEVICE uint8; kv_scale DEVICE float32; out DEVICE bf16.
 * As in cp_attention_step the unused slots of each request's last page are cleared (code 0, scale 1).
 * Decodes (<= 8 rows per KV head) stream the fp8 pages straight into fp8 tensor-core MMAs; requests with a
 * prefill chunk have their pages dequantised (exactly) into the library's bf16 scratch pool first and run the
 * bf16 tile path over it.  Errors: CP_ESTATE (context not created with CP_KV_E4M3, no batch), CP_EINVAL, CP_ECUDA;
 * cp_build_batch returns CP_ECAPACITY when the batch needs more scratch pages than max_scratch_pages. */
int cp_attention_step_fp8(cp_ctx* ctx, int32_t layer, const void* q, const void* k_new, const void* v_new,
                          void* kv_cache8, void* kv_scale, void* out, void* cuda_stream);

/* H6: drain the ring of timed steps, oldest first, into rows (HOST, capacity cap);
 * *n_out receives the count.  Waits for the newest recorded step to finish.  The memory
 * features are what cp_set_memory_stats last stored (zeros if never called). */
int cp_latency_table(cp_ctx* ctx, cp_latency_row* rows, int32_t cap, int32_t* n_out);

/* Table 1's four memory features come from the caller's allocator (PyTorch owns device
 * memory here); values in MB, copied into subsequent latency rows. */
int cp_set_memory_stats(cp_ctx* ctx, float gpu_mem_used_mb, float gpu_mem_free_mb,
                        float cuda_allocated_mb, float cuda_reserved_mb);

/* Introspection of the current batch (for tests and the roofline report). */
typedef struct {
    int32_t n_reqs, n_tokens, n_work_items;
    int32_t n_combine_items;     /* split-KV groups of the batch: grid_combine of them are merged by the combine
                                    kernel (chunk tiles), the others (decodes and <= 16-row chunk tails) inside the
                                    attention kernel by the split that arrives last (no launch)                    */
    int32_t n_tc_items;          /* items routed to the tensor-core tile path      */
    int64_t n_partial_rows;      /* workspace rows in use                          */
    int32_t kernels_per_step;    /* kernel launches one cp_attention_step issues (append, attention; the combine
                                    kernel only when grid_combine > 0; the scratch dequantisation for fp8 chunks;
                                    a small decode-only batch over bf16 pages is ONE launch: the attention kernel
                                    appends the new rows and clears the page tails itself)                        */
    int32_t grid_attn, grid_combine;
    double  alg_flops, alg_bytes; /* algorithmic work of ONE layer's step (SURVEY.md 8(d) formulas: FLOPs = 4 D Hq x causal
                                    pairs; bytes = KV once per request and KV head + Q + out + 4 B per page)          */
    int32_t split;               /* 1: tensor-bound batch, runs the SPLIT instantiation of the kernel (both
                                    softmax warpgroups on every chunk tile); 0: dual-lane instantiation */
} cp_batch_info;
int cp_get_batch_info(cp_ctx* ctx, cp_batch_info* info);

/* ---------------------------------------------------------------------------------
 * Host-side scheduler (no GPU).  H0 of SURVEY.md 8(a).  Forms one iteration under a
 * token budget or a target time: decode first, prefills ranked by the
 * aging key K_i = -alpha a_i + beta r_i (Eq. 4) in a max-heap
 * (PAPER.md:101), chunk by Eq. 6-7 (token budget) or Algorithm 1 (LPRS, Eq. 8-11,
 * PAPER.md:165-253), gated by APC (Eq. 12-14).  Readings of silent
 * points: DESIGN.md S1-S14.  Output is bit-identical to oracle/ref_scheduler.py.
 * ------------------------------------------------------------------------------- */
#define CP_MODE_TOKEN_BUDGET 0
#define CP_MODE_LPRS         1
#define CP_PRED_LINEAR       0    /* T_hat = sum_k w[k] z[k], k ascending             */
#define CP_PRED_MLP          1    /* 16->128->64->32->1 ReLU (Table 7)  */

typedef struct {
    double  alpha;          /* > 0, per second of waiting (Eq. 1)                     */
    double  beta;           /* < 0, per remaining prefill token (Eq. 1)               */
    int32_t B_max;          /* hard token budget per round (Eq. 6)                    */
    int32_t S_max;          /* maximum sequences per batch (Eq. 12)                   */
    int32_t mode;           /* CP_MODE_*                                              */
    int32_t apc;            /* 0/1: Active Prefill Control                            */
    int32_t Delta;          /* search granularity (Eq. 8)                             */
    int32_t C_max;          /* configured max active prefills (Eq. 12)                */
    int32_t L_min;          /* minimum effective chunk (Eq. 12-13)                    */
    int32_t block_size;     /* tokens per page                                        */
    int64_t num_blocks;     /* pages in the pool                                      */
    double  T_star;         /* target latency budget, same unit as the predictor      */
    double  lambda_u;       /* underfill penalty (Eq. 10)                             */
    double  lambda_o;       /* overflow penalty, > lambda_u (Eq. 10)                  */
    double  page_mb;        /* MB per page, for the deterministic memory features     */
    int32_t pred_kind;      /* CP_PRED_*                                              */
    int32_t n_pred_weights; /* 16 (linear) or 12673 (MLP)                             */
    const double* pred_weights;   /* HOST, copied                                     */
    const double* feat_mu;        /* HOST [16] or NULL (= 0): z = (x - mu) * inv_sigma */
    const double* feat_inv_sigma; /* HOST [16] or NULL (= 1)                          */
} cp_sched_config;

typedef struct {
    int64_t n_iters;
    int64_t blocked_by_activity_cap;   /* Table 10 */
    int64_t blocked_by_min_chunk;      /* Table 10 */
    int64_t used_pages;
    int32_t n_waiting, n_decoding, n_future;
} cp_sched_stats;

int cp_sched_create(const cp_sched_config* cfg, cp_sched** out);
int cp_sched_destroy(cp_sched* s);
/* Register a request (arrival in integer microseconds).  CP_EINVAL: prompt_len < 1,
 * output_len < 1 or duplicate id; CP_ECAPACITY: can never fit the pool. */
int cp_sched_add_request(cp_sched* s, int64_t req_id, int64_t arrival_us,
                         int32_t prompt_len, int32_t output_len);
/* Form one iteration at clock now_us: decodes first in (arrival_us, req_id) order, then
 * prefill chunks in selection order.  out: HOST array of capacity cap; each
 * block_table pointer stays valid until the next cp_sched_commit / cp_sched_destroy.
 * *n_out == 0 means nothing is runnable (no commit needed; advance the clock to
 * cp_sched_next_arrival).  CP_ESTATE if the previous iteration was not committed,
 * CP_ECAPACITY if cap is too small. */
int cp_sched_next(cp_sched* s, int64_t now_us, cp_req_desc* out, int32_t cap,
                  int32_t* n_out);
/* Advance request states after the iteration ran for iter_us (Eq. 2, requeue, TTFT). */
int cp_sched_commit(cp_sched* s, int64_t iter_us);
int cp_sched_next_arrival(cp_sched* s, int64_t* arrival_us);  /* -1 if none */
int cp_sched_has_work(cp_sched* s, int32_t* has_work);
int cp_sched_get_stats(cp_sched* s, cp_sched_stats* st);
/* Per-request result: TTFT and finish time in us (-1 if not reached yet). */
int cp_sched_request_times(cp_sched* s, int64_t req_id, int64_t* ttft_us,
                           int64_t* finish_us);
/* Exposed for pinning against the reference (pure functions of the config): */
int cp_sched_predict(cp_sched* s, const double* x16, double* t_hat);
int cp_sched_select_chunk(cp_sched* s, int32_t r_i, int32_t ctx_i, int32_t U_t,
                          int32_t n_dec, int64_t sum_ctx, int32_t max_ctx,
                          int32_t pf_tokens, int32_t n_pf, int64_t pf_proc,
                          int32_t pf_proc_max, int32_t* c_star);

/* ---- an entry point that allocates nothing ---------------------------------------------------------------------
 * cp_decode_attention_static: split-KV decode attention (q_len = 1 per request) over a bf16 paged KV pool, for
 * callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it).  It needs no cp_ctx and calls no cudaMalloc / cudaFree / allocating library routine: the split-KV partials
 * (one unnormalised fp32 O row and one (m, l) pair per (request, q head, split)) live in a file-scope static device
 * array of CP_STATIC_SCRATCH_BYTES (about 2 MiB) inside libcp.so, which every GPU that loads the library holds until
 * the process exits.  Operation: the same as cp_attention_step for a decode:
 * row (request j, q head h) attends to keys [0, kv_len[j]) of KV head h / (num_q_heads / num_kv_heads); fp32
 * softmax, bf16 out.  Plain-ALU kernels (one warp per partial row): a convenience path, not the tuned one.
 *
 *   q             DEVICE  bf16 [n_reqs][num_q_heads][head_dim]
 *   kv_cache      DEVICE  bf16 [num_blocks][2][num_kv_heads][block_size][head_dim]   (the layout of cp_attention_step;
 *                 the new token's K/V row must already be in its page: this call appends nothing)
 *   block_tables  DEVICE  int32 [n_reqs][max_pages_per_req]; row j holds the pages of request j, entries past
 *                 ceil(kv_len[j] / block_size) are not read
 *   kv_len        DEVICE  int32 [n_reqs], each >= 1 (keys of the request, the new token included)
 *   n_splits      key-range splits per row, >= 1 (more splits = more parallelism for few long requests)
 *   out           DEVICE  bf16 [n_reqs][num_q_heads][head_dim]
 *   stream        cudaStream_t (NULL = default stream); the call only enqueues two kernels on it
 * Nothing is owned or kept by the library.  kv_len and the page ids are on the device and are NOT checked.
 * Limit: n_reqs * num_q_heads * n_splits <= CP_STATIC_MAX_PARTIAL_ROWS, else CP_ECAPACITY (nothing is launched);
 * head_dim 64 or 128.  Other errors: CP_EINVAL (null pointer, bad shape), CP_ECUDA.
 * The array is shared by ALL calls on a device and keeps the last call's contents.  Every call overwrites each
 * partial it later reads, so nothing needs clearing between calls; but calls that overlap on the GPU (different
 * streams, or several host threads on one device) race on it: serialise them on one stream. */
#define CP_STATIC_MAX_PARTIAL_ROWS 4096
#define CP_STATIC_SCRATCH_BYTES    (CP_STATIC_MAX_PARTIAL_ROWS * (128 * 4 + 8))
int cp_decode_attention_static(const void* q, const void* kv_cache, const int32_t* block_tables,
                               const int32_t* kv_len, int32_t n_reqs, int32_t max_pages_per_req,
                               int32_t num_q_heads, int32_t num_kv_heads, int32_t head_dim,
                               int32_t block_size, float sm_scale, int32_t n_splits, void* out, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* CP_H_ */
