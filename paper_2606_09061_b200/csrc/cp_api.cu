// cp_api.cu -- libcp's C ABI for the GPU path: context, batch packing (H1), the attention
// step launcher (H2-H5) and the latency table (H6).  See include/cp.h for the contract.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <utility>
#include <vector>

#include "cp_internal.h"
#include "cp_kernels_simt.cuh"
#include "cp_kernels_dl.cuh"

using namespace cp;

#define CP_CUDA(call)                                                                     \
    do {                                                                                  \
        cudaError_t e__ = (call);                                                         \
        if (e__ != cudaSuccess) {                                                         \
            cp_set_error("%s:%d %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e__)); \
            return CP_ECUDA;                                                              \
        }                                                                                 \
    } while (0)

namespace {

// Launch with programmatic dependent launch: the kernel may become resident while its predecessor in
// the stream is still running; it calls griddepcontrol.wait before it touches anything the
// predecessor wrote, so only its prologue (and the launch latency) overlaps.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args&&... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr{};
    attr.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr.val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

constexpr int kRing = 4096;           // timed steps kept for cp_latency_table
constexpr int kMetaRing = 4;          // batches whose metadata may be in flight (staging + device copies)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct TimedStep {
    cudaEvent_t start = nullptr, stop = nullptr;
    cp_latency_row row{};
};

}  // namespace

struct cp_ctx {
    cp_config cfg{};
    Shape shape{};
    int n_sm = 148;
    int tq = 32;                       // tokens per Q tile = 128 / G
    bool use_tc = true;                // false only in -DCP_DEBUG_VARIANTS builds with kernel_variant 1 (SIMT cross-check)

    // limits
    size_t max_items = 0, max_combine = 0, meta_cap = 0;
    int64_t max_partial_rows = 0;

    // device
    uint8_t* d_meta[kMetaRing] = {};   // ring: the copy of batch n overlaps the steps of batch n-1
    float* d_part_o = nullptr;
    float2* d_part_ml = nullptr;
    int32_t* d_counter = nullptr;      // persistent-kernel work counter
    int32_t* d_group_cnt = nullptr;    // [max_combine] arrival counters of the groups merged inside the attention kernel (0 between launches)
    // rotary embedding fused into the append (cp_enable_rope); all null / -1 until enabled
    double* d_inv_freq = nullptr;      // [D/2]
    float2* d_rope_cs = nullptr;       // [max_tokens][D/2] (cos, sin) of the current batch's positions
    __nv_bfloat16* d_q_rot = nullptr;  // [max_tokens][Hq][D] rotated Q of the running step
    int64_t rope_table_iter = -1;      // iter the table was computed for
    // pinned staging ring + the library's copy stream.  Slot s = batch number % kMetaRing:
    //   copy_done[s]  (copy stream)      the H2D of the slot's batch has finished
    //   batch_end[s]  (caller's stream)  recorded by the NEXT cp_build_batch: every step of the slot's batch precedes it
    uint8_t* h_stage[kMetaRing] = {};
    cudaEvent_t copy_done[kMetaRing] = {};
    cudaEvent_t batch_end[kMetaRing] = {};
    bool slot_used[kMetaRing] = {};
    int slot = -1;                     // slot of the current batch
    cudaStream_t copy_stream = nullptr;
    cudaStream_t step_stream = nullptr;   // stream of the current batch's most recent step (else of its build)

    // current batch
    bool have_batch = false;
    BatchMeta meta{};
    cp_batch_info info{};
    int64_t iter = -1;
    float feat[CP_NUM_RAW_FEATURES] = {0};
    float mem_stats[4] = {0, 0, 0, 0};
    int32_t n_prefill = 0, n_decode = 0;
    int32_t combine_rows = 0;          // rows (token, head) that have split partials to merge
    bool tensor_bound = false;         // algorithmic FLOPs / 2.25 PF/s > algorithmic bytes / 8 TB/s (nominal B200)

    // latency ring
    std::vector<TimedStep> ring;
    int64_t ring_head = 0, ring_tail = 0;   // [tail, head) are undrained

    // host scratch reused across build_batch calls (no allocation in steady state)
    std::vector<WorkItem> items, sorted;
    std::vector<CombineItem> combines, fused;   // groups merged by combine_kernel / inside the attention kernel (swap kind)
    std::vector<int32_t> bucket, plan, plan_prow, plan_aux, aux, sorted_aux;
#ifdef CP_DEBUG_VARIANTS
    std::vector<uint32_t> page_mark;   // debug builds: page -> number of the last build that named it
    uint32_t mark_epoch = 0;
#endif

    // fp8 pools (cfg.kv_dtype == CP_KV_E4M3): the bf16 scratch pool of the requests with a prefill chunk
    bool kv8 = false;
    __nv_bfloat16* d_scratch = nullptr;
    int64_t max_scratch_pages = 0;
    int32_t scratch_pages = 0;         // in use by the current batch
    std::vector<int32_t> scratch_base, scratch_req;
    // tensor-core path: one TMA descriptor per KV pool pointer (one per layer), encoded once
    std::vector<std::pair<const void*, CUtensorMap>> tmaps;
    void* encode_fn = nullptr;
    bool tc_attr_set = false;
};

extern "C" int cp_create(const cp_config* cfg, cp_ctx** out) {
    if (!cfg || !out) { cp_set_error("cp_create: null argument"); return CP_EINVAL; }
    const int Hq = cfg->num_q_heads, Hkv = cfg->num_kv_heads, D = cfg->head_dim;
    if (Hq < 1 || Hkv < 1 || Hq % Hkv != 0) { cp_set_error("cp_create: Hq must be a multiple of Hkv"); return CP_EINVAL; }
    const int G = Hq / Hkv;
    if (!(G == 1 || G == 2 || G == 4 || G == 8 || G == 16)) { cp_set_error("cp_create: G = Hq/Hkv must be in {1,2,4,8,16}"); return CP_EINVAL; }
    if (!(D == 64 || D == 128)) { cp_set_error("cp_create: head_dim must be 64 or 128"); return CP_EINVAL; }
    if (cfg->block_size != 16) { cp_set_error("cp_create: block_size must be 16"); return CP_EINVAL; }
    if (cfg->kv_dtype != CP_KV_BF16 && cfg->kv_dtype != CP_KV_E4M3) { cp_set_error("cp_create: kv_dtype must be CP_KV_BF16 or CP_KV_E4M3"); return CP_EINVAL; }
    if (cfg->kv_dtype == CP_KV_E4M3 && (D != 128 || G > 16 || cfg->kernel_variant != 0)) { cp_set_error("cp_create: e4m3 pools need head_dim 128"); return CP_EINVAL; }
    if (cfg->reserved != 0 || cfg->max_scratch_pages < 0) { cp_set_error("cp_create: reserved must be 0, max_scratch_pages >= 0"); return CP_EINVAL; }
    if (cfg->num_blocks < 1 || cfg->max_tokens < 1 || cfg->max_reqs < 1 || cfg->max_total_pages < 1 ||
        cfg->num_layers < 1) { cp_set_error("cp_create: limits must be positive"); return CP_EINVAL; }
    if ((int64_t)cfg->num_blocks * 2 * Hkv >= (int64_t)1 << 31) { cp_set_error("cp_create: pool too large for 32-bit slab index"); return CP_EINVAL; }
    // the kernels take max(raw score) * scale as the maximum of the scaled scores
    if (!(cfg->sm_scale > 0.f) || cfg->sm_scale - cfg->sm_scale != 0.f) { cp_set_error("cp_create: sm_scale must be finite and > 0"); return CP_EINVAL; }

    CP_CUDA(cudaSetDevice(cfg->device));
    cp_ctx* c = new cp_ctx();
    c->cfg = *cfg;
    c->shape = Shape{Hq, Hkv, D, cfg->block_size, G, cfg->sm_scale};
    c->tq = 128 / G;
    cudaDeviceProp prop{};
    if (cudaGetDeviceProperties(&prop, cfg->device) == cudaSuccess) c->n_sm = prop.multiProcessorCount;
    // ONE attention kernel (no dispatch, no fallback): refuse anything but an sm_100 device.  Debug builds
    // (-DCP_DEBUG_VARIANTS) additionally accept kernel_variant 1, the SIMT cross-check kernel used for bisecting.
#ifdef CP_DEBUG_VARIANTS
    if (cfg->kernel_variant != 0 && cfg->kernel_variant != 1) { delete c; cp_set_error("cp_create: kernel_variant must be 0 or 1"); return CP_EINVAL; }
    c->use_tc = cfg->kernel_variant == 0;
#else
    if (cfg->kernel_variant != 0) { delete c; cp_set_error("cp_create: kernel_variant must be 0 (other values exist only in -DCP_DEBUG_VARIANTS builds)"); return CP_EINVAL; }
#endif
    if (c->use_tc && prop.major != 10) { delete c; cp_set_error("cp_create: the attention kernel needs an sm_100 device"); return CP_EINVAL; }
    const size_t q_tiles = (size_t)cfg->max_reqs + (size_t)cfg->max_tokens / c->tq + 1;
    c->max_items = q_tiles * Hkv + (size_t)c->n_sm * 16 + 64;
    c->max_combine = q_tiles * Hkv;
    c->max_partial_rows = cfg->max_partial_rows > 0 ? cfg->max_partial_rows
                                                     : (int64_t)4 * cfg->max_tokens * Hq;
    size_t cap = 0;
    cap += align_up(sizeof(int32_t) * (cfg->max_reqs + 1), 16) * 2;      // cu_q, bt_off
    cap += align_up(sizeof(int32_t) * cfg->max_reqs, 16) * 2;            // q_len, ctx_off
    cap += align_up(sizeof(int32_t) * (size_t)cfg->max_total_pages, 16);
    cap += align_up(sizeof(int32_t) * (size_t)cfg->max_tokens, 16);      // tok_req
    c->kv8 = cfg->kv_dtype == CP_KV_E4M3;
    c->max_scratch_pages = c->kv8 ? (cfg->max_scratch_pages > 0 ? cfg->max_scratch_pages : cfg->max_total_pages) : 0;
    if (c->kv8) cap += align_up(sizeof(int32_t) * cfg->max_reqs, 16) + align_up(sizeof(int32_t) * (size_t)c->max_scratch_pages, 16);
    cap += align_up(sizeof(WorkItem) * c->max_items, 16);
    cap += align_up(sizeof(int32_t) * c->max_items, 16);                 // work_aux
    cap += align_up(sizeof(CombineItem) * c->max_combine, 16);
    c->meta_cap = cap;

    cudaError_t e = cudaSuccess;
    auto chk = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
    for (int i = 0; i < kMetaRing; ++i) chk(cudaMalloc(&c->d_meta[i], cap));
    chk(cudaMalloc(&c->d_part_o, sizeof(float) * (size_t)c->max_partial_rows * D));
    chk(cudaMalloc(&c->d_part_ml, sizeof(float2) * (size_t)c->max_partial_rows));
    chk(cudaMalloc(&c->d_counter, sizeof(int32_t) * 4));
    chk(cudaMalloc(&c->d_group_cnt, sizeof(int32_t) * c->max_combine));
    if (e == cudaSuccess) chk(cudaMemset(c->d_group_cnt, 0, sizeof(int32_t) * c->max_combine));
    if (c->kv8) chk(cudaMalloc(&c->d_scratch, sizeof(__nv_bfloat16) * (size_t)c->max_scratch_pages * 2 * Hkv * cfg->block_size * D));
    chk(cudaMemset(c->d_counter, 0, sizeof(int32_t) * 4));
    for (int i = 0; i < kMetaRing; ++i) {
        chk(cudaMallocHost(&c->h_stage[i], cap));
        chk(cudaEventCreateWithFlags(&c->copy_done[i], cudaEventDisableTiming));
        chk(cudaEventCreateWithFlags(&c->batch_end[i], cudaEventDisableTiming));
    }
    chk(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    c->ring.resize(kRing);
    for (auto& t : c->ring) {
        chk(cudaEventCreate(&t.start));
        chk(cudaEventCreate(&t.stop));
    }
    if (e != cudaSuccess) {
        cp_set_error("cp_create: CUDA allocation failed: %s", cudaGetErrorString(e));
        cp_destroy(c);
        return CP_ECUDA;
    }
#ifdef CP_DEBUG_VARIANTS
    c->page_mark.assign((size_t)cfg->num_blocks, 0);
#endif
    c->items.reserve(c->max_items);
    c->sorted.reserve(c->max_items);
    c->combines.reserve(c->max_combine);
    c->fused.reserve(c->max_combine);
    c->plan_aux.reserve(q_tiles * Hkv);
    c->aux.reserve(c->max_items);
    c->sorted_aux.reserve(c->max_items);
    c->plan.reserve(2 * q_tiles);
    c->plan_prow.reserve(q_tiles * Hkv);
    *out = c;
    return CP_OK;
}

extern "C" int cp_destroy(cp_ctx* c) {
    if (!c) return CP_OK;
    cudaSetDevice(c->cfg.device);
    cudaDeviceSynchronize();
    for (int i = 0; i < kMetaRing; ++i) cudaFree(c->d_meta[i]);
    cudaFree(c->d_part_o);
    cudaFree(c->d_part_ml);
    cudaFree(c->d_counter);
    cudaFree(c->d_group_cnt);
    cudaFree(c->d_scratch);
    cudaFree(c->d_inv_freq);
    cudaFree(c->d_rope_cs);
    cudaFree(c->d_q_rot);
    for (int i = 0; i < kMetaRing; ++i) {
        if (c->h_stage[i]) cudaFreeHost(c->h_stage[i]);
        if (c->copy_done[i]) cudaEventDestroy(c->copy_done[i]);
        if (c->batch_end[i]) cudaEventDestroy(c->batch_end[i]);
    }
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    for (auto& t : c->ring) {
        if (t.start) cudaEventDestroy(t.start);
        if (t.stop) cudaEventDestroy(t.stop);
    }
    delete c;
    return CP_OK;
}

// ------------------------------------------------------------------------------------
// H1: cp_build_batch -- validate, plan the work list, pack, one async H2D copy.
// ------------------------------------------------------------------------------------
extern "C" int cp_build_batch(cp_ctx* c, const cp_req_desc* reqs, int32_t n_reqs, void* stream_) {
    if (!c || (!reqs && n_reqs > 0) || n_reqs < 0) { cp_set_error("cp_build_batch: bad argument"); return CP_EINVAL; }
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const Shape& sh = c->shape;
    const int B = sh.B, G = sh.G;
    if (n_reqs > c->cfg.max_reqs) { cp_set_error("cp_build_batch: %d requests > max_reqs %d", n_reqs, c->cfg.max_reqs); return CP_ECAPACITY; }

    // ---- validate + totals ------------------------------------------------------------
    int64_t T = 0, P = 0, total_tiles[2] = {0, 0};      // key tiles per item kind (tile, swap)
    float f_pf_tokens = 0, f_dec = 0, f_sum_ctx = 0, f_max_ctx = 0, f_pf_proc = 0, f_pf_proc_max = 0;
    int32_t n_prefill = 0, n_decode = 0;
    double alg_pairs = 0, alg_keys = 0;
#ifdef CP_DEBUG_VARIANTS
    const uint32_t epoch = ++c->mark_epoch;
#endif
    for (int j = 0; j < n_reqs; ++j) {
        const cp_req_desc& r = reqs[j];
        if (r.q_len < 1 || r.ctx_off < 0 || r.n_blocks < 0 || (!r.block_table && r.n_blocks > 0)) {
            cp_set_error("cp_build_batch: request %d: q_len %d ctx_off %d n_blocks %d", j, r.q_len, r.ctx_off, r.n_blocks);
            return CP_EINVAL;
        }
        const int64_t kv_len = (int64_t)r.ctx_off + r.q_len;
        alg_pairs += (double)r.q_len * r.ctx_off + 0.5 * r.q_len * ((double)r.q_len + 1);   // causal (query, key) pairs
        alg_keys += (double)kv_len;
        if ((int64_t)r.n_blocks * B < kv_len || kv_len > INT32_MAX) {
            cp_set_error("cp_build_batch: request %d: block table covers %lld < %lld tokens", j,
                         (long long)r.n_blocks * B, (long long)kv_len);
            return CP_EINVAL;
        }
        const int used_pages = (int)((kv_len + B - 1) / B);
        for (int p = 0; p < used_pages; ++p) {
            if (r.block_table[p] < 0 || r.block_table[p] >= c->cfg.num_blocks) {
                cp_set_error("cp_build_batch: request %d: page id %d out of range", j, r.block_table[p]);
                return CP_EINVAL;
            }
#ifdef CP_DEBUG_VARIANTS
            if (c->page_mark[r.block_table[p]] == epoch) {
                cp_set_error("cp_build_batch: request %d: page id %d appears twice in the batch", j, r.block_table[p]);
                return CP_EINVAL;
            }
            c->page_mark[r.block_table[p]] = epoch;
#endif
        }
        T += r.q_len;
        P += used_pages;
        if (r.q_len == 1 && !(r.flags & CP_REQ_PREFILL)) {
            ++n_decode; f_dec += 1; f_sum_ctx += (float)(r.ctx_off + 1);
            f_max_ctx = std::max(f_max_ctx, (float)(r.ctx_off + 1));
        } else {
            ++n_prefill; f_pf_tokens += (float)r.q_len; f_pf_proc += (float)r.ctx_off;
            f_pf_proc_max = std::max(f_pf_proc_max, (float)r.ctx_off);
        }
    }
    // SURVEY.md 8(d) formulas: FLOPs = 4 D Hq pairs; bytes = KV once per request and KV head + Q + out.  A batch
    // that is tensor-bound at the nominal B200 rates runs the SPLIT instantiation of the kernel: both softmax
    // warpgroups of a CTA work on every chunk tile (cp_kernels_dl.cuh).
    bool tensor_bound;
    {
        const double flops = 4.0 * sh.D * sh.Hq * alg_pairs;
        const double bytes = 2.0 * alg_keys * sh.Hkv * sh.D * 2 + 2.0 * (double)T * sh.Hq * sh.D * 2;
        tensor_bound = c->use_tc && flops / 2.25e15 > bytes / 8e12;
    }
    if (c->kv8) tensor_bound = false;                    // fp8 pools: always the dual-lane instantiation
    const int TQ = c->tq;                                // tokens per tile-kind item
    const int swap_rows = c->kv8 ? 8 : 16;               // rows of a swap-kind item (fp8: hi / lo codes share the 16 B rows)
    for (int j = 0; j < n_reqs; ++j) {
        const cp_req_desc& r = reqs[j];
        for (int q0 = 0; q0 < r.q_len; q0 += TQ) {
            const int qt = std::min(TQ, r.q_len - q0);
            const int64_t lim = (int64_t)r.ctx_off + q0 + qt;
            const int kind = (c->use_tc && qt * G <= swap_rows && sh.D == 128) ? kKindSwap : kKindTile;
            total_tiles[kind] += (lim + kKeyTile - 1) / kKeyTile * sh.Hkv;
        }
    }
    if (T > c->cfg.max_tokens) { cp_set_error("cp_build_batch: %lld tokens > max_tokens %d", (long long)T, c->cfg.max_tokens); return CP_ECAPACITY; }
    if (P > c->cfg.max_total_pages) { cp_set_error("cp_build_batch: %lld pages > max_total_pages %lld", (long long)P, (long long)c->cfg.max_total_pages); return CP_ECAPACITY; }

    // ---- plan: split long key ranges so the persistent grid stays balanced ---------------
    // An item is never longer than (total key tiles of the batch) / (n_sm * P), so the LPT-ordered
    // dynamic schedule ends with a short tail.  Splitting a chunk tile is expensive (a 64 KiB fp32
    // partial per split, a second pipeline fill, the combine pass), so tile-kind items are split only
    // when LPT needs it (P = 1: no item above the mean load of an SM); decode items cost 2 KiB per
    // split, and a decode-only batch should give each of the two lanes of an SM an item (P = 2).
    // Measured on B200: P = 12 for both kinds cost 14 % on the chunks of
    // configs[2] and 20 % on configs[1].
    int per_sm[2] = {1, 2};
    if (!c->use_tc) per_sm[0] = per_sm[1] = 12;                   // SIMT cross-check kernel (debug builds): one CTA per item
    int chunk_of[2];
    for (int k = 0; k < 2; ++k) {
        const int64_t total = total_tiles[0] + total_tiles[1];     // the lanes share the SMs: mean load of the whole batch
        const int64_t per = (int64_t)c->n_sm * per_sm[k];
        chunk_of[k] = (int)std::min<int64_t>(1 << 20, std::max<int64_t>(1, (total + per - 1) / per));
    }
    // Few decode items per lane: the NUMBER OF ROUNDS a lane runs decides the time, not the mean load.  With items no
    // longer than the mean load, per-request rounding leaves slightly more items than lanes (12 long decodes: 328 items
    // on 296 lanes), and the lanes that draw a second item finish a whole item late while the rest of the GPU idles.
    // So among chunk lengths from the mean load up to twice that (coarser only: never more splits or workspace than
    // before), take the one with the smallest rounds x (chunk + per-item start-up, ~2 tiles); a round counts as full at
    // 15/16 of the lanes (measured optimum: 264 items beat 288 and 296 on 296 lanes).  B200, 8B shape: 12 long decodes
    // 169 -> 153 us, 6 x 30 K tokens 142 -> 126, 14 decodes of the trace's context mix 68 -> 58, decode-only rounds of
    // the configs[4] trace 1342 -> 1190 us per 32 layers (p50); batches with many items per lane are unchanged.
    if (c->use_tc && total_tiles[1] > 0) {
        const int64_t lanes = (int64_t)c->n_sm * (total_tiles[0] == 0 ? 2 : 1);
        auto items_at = [&](int chunk) {
            int64_t n = 0;
            for (int j = 0; j < n_reqs; ++j) {
                const cp_req_desc& r = reqs[j];
                for (int q0 = 0; q0 < r.q_len; q0 += TQ) {
                    const int qt = std::min(TQ, r.q_len - q0);
                    if (qt * G > swap_rows || sh.D != 128) continue;
                    const int n_tiles = (int)(((int64_t)r.ctx_off + q0 + qt + kKeyTile - 1) / kKeyTile);
                    n += (int64_t)((n_tiles + chunk - 1) / chunk) * sh.Hkv;
                }
            }
            return n;
        };
        const int c0 = chunk_of[1];
        if (c0 < (1 << 19) && items_at(c0) <= 3 * lanes) {
            const int64_t fill = std::max<int64_t>(1, lanes * 15 / 16);
            int best = c0;
            int64_t best_cost = ((items_at(c0) + fill - 1) / fill) * (c0 + 2);
            for (int k = 1; k <= 16; ++k) {
                const int chunk = c0 + (int)(((int64_t)c0 * k + 15) / 16);
                const int64_t cost = ((items_at(chunk) + fill - 1) / fill) * (chunk + 2);
                if (cost < best_cost) { best_cost = cost; best = chunk; }
            }
            chunk_of[1] = best;
        }
    }
    int64_t partial_rows = 0;
    for (int attempt = 0;; ++attempt) {
        c->items.clear();
        c->aux.clear();
        c->combines.clear();
        c->fused.clear();
        partial_rows = 0;
        int64_t tok = 0;
        bool overflow = false;
        for (int j = 0; j < n_reqs && !overflow; ++j) {
            const cp_req_desc& r = reqs[j];
            // pass 1: per (q tile, KV head) group, reserve the split workspace and the combine item
            const int nq = (r.q_len + TQ - 1) / TQ;
            c->plan.resize((size_t)nq * 2);                          // [qi] = {n_splits, tps}
            c->plan_prow.resize((size_t)nq * sh.Hkv);
            c->plan_aux.resize((size_t)nq * sh.Hkv);
            int max_splits = 0;
            for (int qi = 0; qi < nq && !overflow; ++qi) {
                const int q0 = qi * TQ, qt = std::min(TQ, r.q_len - q0), rows = qt * G;
                const int lim = r.ctx_off + q0 + qt;                 // causal limit of the last row
                const int n_tiles = (lim + kKeyTile - 1) / kKeyTile;
                const int chunk_tiles = chunk_of[(c->use_tc && rows <= swap_rows && sh.D == 128) ? kKindSwap : kKindTile];
                const int n_splits = (n_tiles + chunk_tiles - 1) / chunk_tiles;
                c->plan[2 * qi] = n_splits;
                c->plan[2 * qi + 1] = (n_tiles + n_splits - 1) / n_splits;
                max_splits = std::max(max_splits, n_splits);
                // split groups of the swap kind are merged inside the attention kernel (the last split to arrive
                // does it), the others by combine_kernel
                const bool fuse = c->use_tc && rows <= swap_rows && sh.D == 128;
                for (int g = 0; g < sh.Hkv; ++g) {
                    int32_t prow = -1, aux = -1;
                    if (n_splits > 1) {
                        prow = (int32_t)partial_rows;
                        partial_rows += (int64_t)n_splits * rows;
                        if (partial_rows > c->max_partial_rows || partial_rows > INT32_MAX ||
                            c->combines.size() + c->fused.size() >= c->max_combine) { overflow = true; break; }
                        const CombineItem ci{(int32_t)(tok + q0), qt, g, n_splits, prow, 0, {0, 0}};
                        if (fuse) { aux = (int32_t)c->fused.size(); c->fused.push_back(ci); }
                        else c->combines.push_back(ci);
                    }
                    c->plan_prow[(size_t)qi * sh.Hkv + g] = prow;
                    c->plan_aux[(size_t)qi * sh.Hkv + g] = aux;
                }
                if (c->items.size() + (size_t)n_splits * sh.Hkv > c->max_items) overflow = true;
            }
            // pass 2: emit in (KV head, split, q tile) order, so that the q tiles of a chunk that read
            // the same K/V range sit next to each other in the work list, start together on
            // neighbouring SMs and share those K/V tiles in L2 (one DRAM fetch for all of them)
            size_t emitted = 0;
            for (int g = 0; g < sh.Hkv && !overflow; ++g)
                for (int s = 0; s < max_splits && !overflow; ++s)
                    for (int qi = 0; qi < nq; ++qi) {
                        if (s >= c->plan[2 * qi]) continue;
                        const int q0 = qi * TQ, qt = std::min(TQ, r.q_len - q0), rows = qt * G;
                        const int lim = r.ctx_off + q0 + qt, tps = c->plan[2 * qi + 1];
                        const int kind = (c->use_tc && rows <= swap_rows && sh.D == 128) ? kKindSwap : kKindTile;
                        const int32_t prow = c->plan_prow[(size_t)qi * sh.Hkv + g];
                        if (c->items.size() >= c->max_items) { overflow = true; break; }
                        c->items.push_back(WorkItem{j, g, q0, qt, s * tps * kKeyTile, std::min(lim, (s + 1) * tps * kKeyTile),
                                                    prow < 0 ? -1 : prow + s * rows, kind});
                        c->aux.push_back(c->plan_aux[(size_t)qi * sh.Hkv + g]);
                        ++emitted;
                    }
            (void)emitted;
            tok += r.q_len;
        }
        if (!overflow) break;
        if (chunk_of[0] >= (1 << 20) && chunk_of[1] >= (1 << 20)) { cp_set_error("cp_build_batch: work list does not fit the limits of cp_create"); return CP_ECAPACITY; }
        chunk_of[0] = std::min(1 << 20, chunk_of[0] * 2);            // coarser splits need less workspace
        chunk_of[1] = std::min(1 << 20, chunk_of[1] * 2);
    }

    // ---- LPT order: bucket sort by descending number of key tiles.  The dual-lane kernel takes the
    // tile-kind items first and the swap-kind items after them (two lists, one array).
    const size_t n_items = c->items.size();
    int max_cost = 0;
    int32_t n_tile_items = 0;
    // cost = key tiles, in steps of 4: LPT needs no finer order, and items of nearly equal length keep
    // their emission order (the L2-sharing neighbourhoods above)
    auto cost_of = [](const WorkItem& w) { return (w.kv_end - w.kv_begin + 4 * kKeyTile - 1) / (4 * kKeyTile); };
    for (const WorkItem& w : c->items) { max_cost = std::max(max_cost, cost_of(w)); n_tile_items += w.kind == kKindTile; }
    const size_t kind_stride = c->use_tc ? (size_t)max_cost + 1 : 0;
    auto bucket_of = [&](const WorkItem& w) { return (w.kind == kKindSwap ? kind_stride : 0) + (size_t)(max_cost - cost_of(w)); };
    c->bucket.assign(kind_stride + (size_t)max_cost + 2, 0);
    for (const WorkItem& w : c->items) ++c->bucket[bucket_of(w) + 1];
    for (size_t i = 1; i < c->bucket.size(); ++i) c->bucket[i] += c->bucket[i - 1];
    c->sorted.resize(n_items);
    c->sorted_aux.resize(n_items);
    for (size_t i = 0; i < n_items; ++i) {
        const size_t pos = c->bucket[bucket_of(c->items[i])]++;
        c->sorted[pos] = c->items[i];
        c->sorted_aux[pos] = c->aux[i];
    }

    // ---- pack into pinned staging ------------------------------------------------------------
    // the batch that ends here: every step it will ever run has been enqueued on step_stream by now
    if (c->slot >= 0) CP_CUDA(cudaEventRecord(c->batch_end[c->slot], c->step_stream));
    const int si = (c->slot + 1) % kMetaRing;
    // staging slot si was last used kMetaRing batches ago: its copy finished long since; the host waits here
    // only when it runs more than kMetaRing - 1 batches ahead of the device (include/cp.h)
    if (c->slot_used[si]) CP_CUDA(cudaEventSynchronize(c->copy_done[si]));
    uint8_t* h = c->h_stage[si];
    size_t off = 0;
    auto place = [&](size_t bytes) { size_t o = off; off += align_up(bytes, 16); return o; };
    const size_t o_cu = place(sizeof(int32_t) * (n_reqs + 1));
    const size_t o_ql = place(sizeof(int32_t) * n_reqs);
    const size_t o_co = place(sizeof(int32_t) * n_reqs);
    const size_t o_bo = place(sizeof(int32_t) * (n_reqs + 1));
    const size_t o_bt = place(sizeof(int32_t) * (size_t)P);
    const size_t o_tr = place(sizeof(int32_t) * (size_t)T);
    const size_t o_wk = place(sizeof(WorkItem) * n_items);
    const size_t o_wa = place(sizeof(int32_t) * n_items);
    const size_t o_cb = place(sizeof(CombineItem) * (c->combines.size() + c->fused.size()));      // [combine_kernel's | fused]
    // fp8 pools: requests with a tile-kind item get their pages dequantised into the scratch pool, contiguously
    size_t o_sb = 0, o_sr = 0;
    if (c->kv8) {
        c->scratch_base.assign((size_t)n_reqs, -1);
        c->scratch_req.clear();
        for (const WorkItem& w : c->items)
            if (w.kind == kKindTile && c->scratch_base[w.req] < 0) c->scratch_base[w.req] = 0;      // mark
        int64_t used = 0;
        for (int j = 0; j < n_reqs; ++j) {
            if (c->scratch_base[j] < 0) continue;
            const int used_pages = (int)(((int64_t)reqs[j].ctx_off + reqs[j].q_len + B - 1) / B);
            if (used + used_pages > c->max_scratch_pages) {
                cp_set_error("cp_build_batch: the prefill chunks of this batch need more than max_scratch_pages = %lld scratch pages",
                             (long long)c->max_scratch_pages);
                return CP_ECAPACITY;
            }
            c->scratch_base[j] = (int32_t)used;
            c->scratch_req.insert(c->scratch_req.end(), (size_t)used_pages, j);
            used += used_pages;
        }
        o_sb = place(sizeof(int32_t) * n_reqs);
        o_sr = place(sizeof(int32_t) * c->scratch_req.size());
    }
    if (off > c->meta_cap) { cp_set_error("cp_build_batch: metadata %zu B > capacity %zu B", off, c->meta_cap); return CP_ECAPACITY; }
    int32_t* cu = reinterpret_cast<int32_t*>(h + o_cu);
    int32_t* ql = reinterpret_cast<int32_t*>(h + o_ql);
    int32_t* co = reinterpret_cast<int32_t*>(h + o_co);
    int32_t* bo = reinterpret_cast<int32_t*>(h + o_bo);
    int32_t* bt = reinterpret_cast<int32_t*>(h + o_bt);
    int32_t* tr = reinterpret_cast<int32_t*>(h + o_tr);
    cu[0] = 0;
    bo[0] = 0;
    for (int j = 0; j < n_reqs; ++j) {
        const cp_req_desc& r = reqs[j];
        const int used_pages = (int)(((int64_t)r.ctx_off + r.q_len + B - 1) / B);
        ql[j] = r.q_len;
        co[j] = r.ctx_off;
        cu[j + 1] = cu[j] + r.q_len;
        bo[j + 1] = bo[j] + used_pages;
        std::memcpy(bt + bo[j], r.block_table, sizeof(int32_t) * used_pages);
        for (int i = 0; i < r.q_len; ++i) tr[cu[j] + i] = j;
    }
    std::memcpy(h + o_wk, c->sorted.data(), sizeof(WorkItem) * n_items);
    std::memcpy(h + o_wa, c->sorted_aux.data(), sizeof(int32_t) * n_items);
    {   // prefix sums of the groups' row counts: the combine kernel maps one warp to one row
        int32_t rows = 0;
        for (CombineItem& ci : c->combines) { ci.row_base = rows; rows += ci.q_tokens * G; }
        c->combine_rows = rows;
    }
    std::memcpy(h + o_cb, c->combines.data(), sizeof(CombineItem) * c->combines.size());
    std::memcpy(h + o_cb + sizeof(CombineItem) * c->combines.size(), c->fused.data(), sizeof(CombineItem) * c->fused.size());
    if (c->kv8) {
        std::memcpy(h + o_sb, c->scratch_base.data(), sizeof(int32_t) * n_reqs);
        std::memcpy(h + o_sr, c->scratch_req.data(), sizeof(int32_t) * c->scratch_req.size());
        c->scratch_pages = (int32_t)c->scratch_req.size();
    }

    // the copy runs on the library's own stream, next to the previous batch's steps; it waits only for the
    // steps that read this device slot kMetaRing batches ago, and the caller's stream waits for the copy
    uint8_t* d_meta = c->d_meta[si];
    if (c->slot_used[si]) CP_CUDA(cudaStreamWaitEvent(c->copy_stream, c->batch_end[si], 0));
    if (off > 0) CP_CUDA(cudaMemcpyAsync(d_meta, h, off, cudaMemcpyHostToDevice, c->copy_stream));
    CP_CUDA(cudaEventRecord(c->copy_done[si], c->copy_stream));
    CP_CUDA(cudaStreamWaitEvent(stream, c->copy_done[si], 0));
    c->slot_used[si] = true;
    c->slot = si;
    c->step_stream = stream;

    BatchMeta& m = c->meta;
    m.cu_q = reinterpret_cast<const int32_t*>(d_meta + o_cu);
    m.q_len = reinterpret_cast<const int32_t*>(d_meta + o_ql);
    m.ctx_off = reinterpret_cast<const int32_t*>(d_meta + o_co);
    m.bt_off = reinterpret_cast<const int32_t*>(d_meta + o_bo);
    m.block_table = reinterpret_cast<const int32_t*>(d_meta + o_bt);
    m.tok_req = reinterpret_cast<const int32_t*>(d_meta + o_tr);
    m.work = reinterpret_cast<const WorkItem*>(d_meta + o_wk);
    m.work_aux = reinterpret_cast<const int32_t*>(d_meta + o_wa);
    m.combine = reinterpret_cast<const CombineItem*>(d_meta + o_cb);
    m.scratch_base = c->kv8 ? reinterpret_cast<const int32_t*>(d_meta + o_sb) : nullptr;
    m.scratch_req = c->kv8 ? reinterpret_cast<const int32_t*>(d_meta + o_sr) : nullptr;
    m.n_reqs = n_reqs;
    m.n_tokens = (int32_t)T;
    m.n_work = (int32_t)n_items;
    m.n_combine = (int32_t)c->combines.size();
    m.n_tile = n_tile_items;

    int32_t n_tc = 0;
    if (c->use_tc) n_tc = (int32_t)n_items;
    c->info = cp_batch_info{n_reqs, (int32_t)T, (int32_t)n_items, (int32_t)(c->combines.size() + c->fused.size()), n_tc,
                            partial_rows, 0, 0, 0,
                            4.0 * sh.D * sh.Hq * alg_pairs,
                            2.0 * alg_keys * sh.Hkv * (c->kv8 ? sh.D + 4.0 : sh.D * 2.0) + 2.0 * (double)T * sh.Hq * sh.D * 2 + 4.0 * (double)P,
                            tensor_bound ? 1 : 0};
    c->feat[0] = f_pf_tokens; c->feat[1] = f_dec; c->feat[2] = (float)n_reqs; c->feat[3] = f_sum_ctx;
    c->feat[4] = f_max_ctx; c->feat[5] = f_pf_proc; c->feat[6] = f_pf_proc_max;
    c->n_prefill = n_prefill;
    c->n_decode = n_decode;
    c->tensor_bound = tensor_bound;
    c->have_batch = true;
    ++c->iter;
    if (c->d_rope_cs && T > 0) {       // positions changed: (cos, sin) table of this batch, same stream as the copy
        const int half = sh.D / 2;
        const int grid = (int)std::min<int64_t>((T * half + 255) / 256, (int64_t)c->n_sm * 8);
        rope_table_kernel<<<grid, 256, 0, stream>>>(m, half, c->d_inv_freq, c->d_rope_cs);
        CP_CUDA(cudaGetLastError());
    }
    c->rope_table_iter = c->d_rope_cs ? c->iter : -1;
    return CP_OK;
}

// N2: rotary embedding.  Allocates its workspace here (a set-up call, like cp_create).
extern "C" int cp_enable_rope(cp_ctx* c, const double* inv_freq) {
    if (!c || !inv_freq) { cp_set_error("cp_enable_rope: null argument"); return CP_EINVAL; }
    const Shape& sh = c->shape;
    const int half = sh.D / 2;
    for (int i = 0; i < half; ++i)
        if (!(inv_freq[i] == inv_freq[i]) || inv_freq[i] - inv_freq[i] != 0.0) {
            cp_set_error("cp_enable_rope: inv_freq[%d] is not finite", i);
            return CP_EINVAL;
        }
    CP_CUDA(cudaSetDevice(c->cfg.device));
    if (!c->d_inv_freq) {
        double* f = nullptr; float2* cs = nullptr; __nv_bfloat16* qr = nullptr;
        cudaError_t e = cudaMalloc(&f, sizeof(double) * half);
        if (e == cudaSuccess) e = cudaMalloc(&cs, sizeof(float2) * (size_t)c->cfg.max_tokens * half);
        if (e == cudaSuccess) e = cudaMalloc(&qr, sizeof(__nv_bfloat16) * (size_t)c->cfg.max_tokens * sh.Hq * sh.D);
        if (e != cudaSuccess) {
            cudaFree(f); cudaFree(cs); cudaFree(qr);
            cp_set_error("cp_enable_rope: CUDA allocation failed: %s", cudaGetErrorString(e));
            return CP_ECUDA;
        }
        c->d_inv_freq = f; c->d_rope_cs = cs; c->d_q_rot = qr;
    }
    CP_CUDA(cudaDeviceSynchronize());                       // no step may still be reading the old table
    CP_CUDA(cudaMemcpy(c->d_inv_freq, inv_freq, sizeof(double) * half, cudaMemcpyHostToDevice));
    c->rope_table_iter = -1;                                // the current batch (if any) has no table yet
    return CP_OK;
}

// ------------------------------------------------------------------------------------
// H2-H5: cp_attention_step
// ------------------------------------------------------------------------------------
#ifdef CP_DEBUG_VARIANTS
template <int D>
static int launch_simt(cp_ctx* c, const __nv_bfloat16* q, const __nv_bfloat16* cache,
                       __nv_bfloat16* out, cudaStream_t stream) {
    const BatchMeta& m = c->meta;
    if (m.n_work > 0) {
        attn_simt_kernel<D><<<m.n_work, 128, 0, stream>>>(m, c->shape, q, cache, out, c->d_part_o, c->d_part_ml);
        CP_CUDA(cudaGetLastError());
    }
    if (m.n_combine > 0) {
        combine_kernel<D><<<(c->combine_rows + 3) / 4, 128, 0, stream>>>(m, c->shape, c->d_part_o, c->d_part_ml, out);
        CP_CUDA(cudaGetLastError());
    }
    return CP_OK;
}
#endif

typedef CUresult (*cuTensorMapEncodeTiled_t)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                             const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                             CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                             CUtensorMapFloatOOBfill);

// TMA descriptor of one layer's KV pool (slab = (block, K|V, kv head)), 128-byte swizzle.
// kind 0: a bf16 pool of n_pages pages; kind 1: an e4m3 pool (one box = the 16 x 128 B codes of a slab).
static int get_tmap(cp_ctx* c, void* kv_cache, const CUtensorMap** out, int kind = 0, int64_t n_pages = 0) {
    if (n_pages == 0) n_pages = c->cfg.num_blocks;
    const void* key = static_cast<const uint8_t*>(kv_cache) + kind;     // pools are 16-byte aligned: the low bit tags the kind
    for (auto& e : c->tmaps)
        if (e.first == key) { *out = &e.second; return CP_OK; }
    if (!c->encode_fn) {
        cudaDriverEntryPointQueryResult qres;
        CP_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &c->encode_fn, cudaEnableDefault, &qres));
        if (qres != cudaDriverEntryPointSuccess || !c->encode_fn) {
            cp_set_error("cuTensorMapEncodeTiled not available from the driver");
            return CP_ECUDA;
        }
    }
    const Shape& sh = c->shape;
    CUtensorMap m;
    if (kind == 1) {
        // e4m3 pool: 3-D {D bytes, 16 slots, slabs}; a box = one slab = 16 rows of 128 B = two 8-row swizzle groups
        const cuuint64_t dims[3] = {(cuuint64_t)sh.D, 16, (cuuint64_t)n_pages * 2 * sh.Hkv};
        const cuuint64_t strides[2] = {(cuuint64_t)sh.D, (cuuint64_t)sh.D * 16};
        const cuuint32_t box[3] = {(cuuint32_t)sh.D, 16, 1};
        const cuuint32_t estr[3] = {1, 1, 1};
        CUresult r = reinterpret_cast<cuTensorMapEncodeTiled_t>(c->encode_fn)(
            &m, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, kv_cache, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { cp_set_error("cuTensorMapEncodeTiled (e4m3 pool) failed: %d", (int)r); return CP_ECUDA; }
        if (c->tmaps.size() >= 256) c->tmaps.clear();
        c->tmaps.emplace_back(key, m);
        *out = &c->tmaps.back().second;
        return CP_OK;
    }
    // 5-D view of the pool so that ONE box = one whole (block, K|V, head) slab of 16 tokens x D:
    //   d0 64 elements (one 128-byte half-row)     d1 8 tokens of a row group (stride D*2)
    //   d2 D/64 halves of a row (stride 128 B)     d3 2 row groups (stride 8*D*2)
    //   d4 slab index (stride 16*D*2)
    // The box lands in smem as [row group][half][8 rows][128 B]: 8-row groups of each half are
    // D/64 KiB apart for the whole 128-key tile, which is a legal UMMA SBO (see cp_kernels_dl.cuh).
    const cuuint64_t rowb = (cuuint64_t)sh.D * 2;
    const cuuint64_t dims[5] = {64, 8, (cuuint64_t)sh.D / 64, 2, (cuuint64_t)n_pages * 2 * sh.Hkv};
    const cuuint64_t strides[4] = {rowb, 128, 8 * rowb, 16 * rowb};
    const cuuint32_t box[5] = {64, 8, (cuuint32_t)sh.D / 64, 2, 1};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    CUresult r = reinterpret_cast<cuTensorMapEncodeTiled_t>(c->encode_fn)(
        &m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, kv_cache, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
        CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { cp_set_error("cuTensorMapEncodeTiled failed: %d", (int)r); return CP_ECUDA; }
    if (c->tmaps.size() >= 256) c->tmaps.clear();
    c->tmaps.emplace_back(key, m);
    *out = &c->tmaps.back().second;
    return CP_OK;
}

// kv_scale != nullptr: kv_cache is an e4m3 pool (D = 128), chunk tiles read the library's bf16 scratch pool
// k_new_fused / v_new_fused / fused: H2 runs inside the attention kernel (decode-only batches over bf16 pages)
template <int D>
static int launch_tc_d(cp_ctx* c, const __nv_bfloat16* q, void* kv_cache, const float* kv_scale, __nv_bfloat16* out,
                       cudaStream_t stream, int* launches, bool fused, const void* k_new_fused, const void* v_new_fused) {
    const BatchMeta& m = c->meta;
    const CUtensorMap* tmap = nullptr;
    const CUtensorMap* tmap8 = nullptr;
    int rc = kv_scale ? get_tmap(c, c->d_scratch, &tmap, 0, c->max_scratch_pages) : get_tmap(c, kv_cache, &tmap);
    if (rc != CP_OK) return rc;
    // (get_tmap may clear its cache when it grows: take the second descriptor's copy before it could move)
    const CUtensorMap tmap_copy = *tmap;
    if (kv_scale) { rc = get_tmap(c, kv_cache, &tmap8, 1); if (rc != CP_OK) return rc; }
    else tmap8 = &tmap_copy;
    if (!c->tc_attr_set) {
        CP_CUDA(cudaFuncSetAttribute(dl::attn_dl_kernel<D, false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dl::Layout<D, false>::kTotal));
        CP_CUDA(cudaFuncSetAttribute(dl::attn_dl_kernel<D, true, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dl::Layout<D, true>::kTotal));
        if constexpr (D == 128) {
            CP_CUDA(cudaFuncSetAttribute(dl::attn_dl_kernel<128, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dl::Layout<128, false>::kTotal));
            CP_CUDA(cudaFuncSetAttribute(dl::attn_dl_kernel<128, false, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dl::Layout<128, false>::kTotal));
        }
        c->tc_attr_set = true;
    }
    if (m.n_work > 0) {
        const int grid = std::min(c->n_sm, m.n_work);
        dl::Params p{m, c->shape, q, out, c->d_part_o, c->d_part_ml, c->d_counter, kv_scale, c->d_group_cnt,
                     static_cast<const uint4*>(k_new_fused), static_cast<const uint4*>(v_new_fused), static_cast<__nv_bfloat16*>(kv_cache)};
        if (kv_scale) {
            if constexpr (D == 128)
                CP_CUDA(launch_pdl(dl::attn_dl_kernel<128, false, false, true>, dim3(grid), dim3(dl::kThreads), dl::Layout<128, false>::kTotal, stream, p, tmap_copy, *tmap8));
        } else
        // Two instantiations of the one kernel, chosen per batch by the SURVEY.md 8(d) roofline formulas: HBM-bound
        // batches run chunk tiles and decode streams side by side (dual lane); tensor-bound batches put both softmax
        // warpgroups on every chunk tile (SPLIT) and move a quarter of the exponentials to the FMA pipe.
        if (fused) {
            if constexpr (D == 128)
                CP_CUDA(launch_pdl(dl::attn_dl_kernel<128, false, false, false, true>, dim3(grid), dim3(dl::kThreads), dl::Layout<128, false>::kTotal, stream, p, tmap_copy, *tmap8));
        } else if (c->tensor_bound)
            CP_CUDA(launch_pdl(dl::attn_dl_kernel<D, true, true, false>, dim3(grid), dim3(dl::kThreadsSplit), dl::Layout<D, true>::kTotal, stream, p, tmap_copy, *tmap8));
        else
            CP_CUDA(launch_pdl(dl::attn_dl_kernel<D, false, false, false>, dim3(grid), dim3(dl::kThreads), dl::Layout<D, false>::kTotal, stream, p, tmap_copy, *tmap8));
        CP_CUDA(cudaGetLastError());
        ++*launches;
        c->info.grid_attn = grid;
    }
    if (m.n_combine > 0) {
        CP_CUDA(launch_pdl(combine_kernel<D>, dim3((c->combine_rows + 3) / 4), dim3(128), 0, stream, m, c->shape,
                           (const float*)c->d_part_o, (const float2*)c->d_part_ml, out));
        ++*launches;
    }
    c->info.grid_combine = m.n_combine;
    return CP_OK;
}

static int launch_tc(cp_ctx* c, const __nv_bfloat16* q, void* kv_cache, const float* kv_scale, __nv_bfloat16* out,
                     cudaStream_t stream, int* launches, bool fused = false, const void* k_new = nullptr, const void* v_new = nullptr) {
    return c->shape.D == 128 ? launch_tc_d<128>(c, q, kv_cache, kv_scale, out, stream, launches, fused, k_new, v_new)
                             : launch_tc_d<64>(c, q, kv_cache, kv_scale, out, stream, launches, false, nullptr, nullptr);
}

// validate the arguments of one layer's step and enqueue its kernels (no events, no latency row)
static int issue_step(cp_ctx* c, int32_t layer, const void* q, const void* k_new, const void* v_new,
                      void* kv_cache, void* out, cudaStream_t stream, bool rope, void* kv_scale, int* launches_out) {
    if (!c) return CP_EINVAL;
    if (!c->have_batch) { cp_set_error("cp_attention_step: no batch built"); return CP_ESTATE; }
    if (c->kv8 != (kv_scale != nullptr)) {
        cp_set_error(c->kv8 ? "this context drives an e4m3 pool: use cp_attention_step_fp8" : "cp_attention_step_fp8: the context was not created with CP_KV_E4M3");
        return CP_ESTATE;
    }
    if (rope) {
        if (!c->d_rope_cs) { cp_set_error("cp_attention_step_rope: cp_enable_rope was not called"); return CP_ESTATE; }
        if (c->rope_table_iter != c->iter) {
            cp_set_error("cp_attention_step_rope: the batch was built before cp_enable_rope");
            return CP_ESTATE;
        }
        if (!k_new) { cp_set_error("cp_attention_step_rope: k_new / v_new must not be NULL"); return CP_EINVAL; }
    }
    if (!q || !kv_cache || !out || ((k_new == nullptr) != (v_new == nullptr)) || layer < 0) {
        cp_set_error("cp_attention_step: bad argument");
        return CP_EINVAL;
    }
    if ((reinterpret_cast<uintptr_t>(q) | reinterpret_cast<uintptr_t>(kv_cache) | reinterpret_cast<uintptr_t>(out) |
         reinterpret_cast<uintptr_t>(k_new) | reinterpret_cast<uintptr_t>(v_new)) & 15) {
        cp_set_error("cp_attention_step: pointers must be 16-byte aligned");
        return CP_EINVAL;
    }
    c->step_stream = stream;
    const BatchMeta& m = c->meta;
    int launches = 0;
    // A small decode-only batch over bf16 pages (no tile-kind item: every request is one swap-kind q tile) needs no
    // append launch: the attention kernel's producers write the new rows and clear the page tails themselves (H2 inside
    // H4).  One kernel per layer instead of two dependent ones -- what a decode round of the configs[4] trace pays per
    // layer: 16-layer submissions, 14 decodes of the trace's context mix 55.8 -> 52.3 us per layer, 14 short decodes
    // 22.8 -> 20.2, 12 long decodes 149.7 -> 147.4, 70 decodes 86.0 -> 85.5.  With thousands of items the producers'
    // extra work per item costs more than the launch it saves (512 decodes: 491 -> 510 us), hence the item limit.
    const bool fused = c->use_tc && !rope && !c->kv8 && c->shape.D == 128 && m.n_tile == 0 && m.n_work > 0 &&
                       m.n_work <= 4 * c->n_sm && !c->tensor_bound;
    if (m.n_tokens > 0) {
        if (fused) {
            // nothing to launch here
        } else if (rope) {
            const Shape& sh = c->shape;
            const int64_t total = (int64_t)m.n_tokens * (sh.Hkv * (sh.D / 8) + (sh.Hkv + sh.Hq) * (sh.D / 16));
            const int grid = (int)std::min<int64_t>((total + 255) / 256, (int64_t)c->n_sm * 8);
            kv_append_rope_kernel<<<grid, 256, 0, stream>>>(m, sh, static_cast<const uint4*>(q),
                                                            static_cast<const uint4*>(k_new),
                                                            static_cast<const uint4*>(v_new), c->d_rope_cs,
                                                            static_cast<__nv_bfloat16*>(kv_cache),
                                                            reinterpret_cast<uint4*>(c->d_q_rot));
            CP_CUDA(cudaGetLastError());
            ++launches;
            q = c->d_q_rot;
        } else if (kv_scale) {
            // quantise the new rows into the e4m3 pages (and clear the page tails), then dequantise the pages of
            // the requests with a prefill chunk into the bf16 scratch pool
            const Shape& sh = c->shape;
            const int64_t total = std::max<int64_t>(k_new ? (int64_t)m.n_tokens * sh.Hkv * 2 * 16 : 0,
                                                    (int64_t)m.n_reqs * 2 * sh.Hkv * (sh.B - 1) * (sh.D / 16));
            const int grid = (int)std::min<int64_t>((total + 255) / 256, (int64_t)c->n_sm * 8);
            kv_append_q8_kernel<<<grid, 256, 0, stream>>>(m, sh, static_cast<const uint4*>(k_new), static_cast<const uint4*>(v_new),
                                                          static_cast<uint8_t*>(kv_cache), static_cast<float*>(kv_scale));
            CP_CUDA(cudaGetLastError());
            ++launches;
            if (c->scratch_pages > 0) {
                const int g2 = (int)std::min<int64_t>(c->scratch_pages, (int64_t)c->n_sm * 8);      // a CTA per scratch page
                kv8_dequant_kernel<<<g2, 256, 0, stream>>>(m, sh, static_cast<const uint8_t*>(kv_cache), static_cast<const float*>(kv_scale),
                                                           c->d_scratch, c->scratch_pages);
                CP_CUDA(cudaGetLastError());
                ++launches;
            }
        } else {
            // k_new == NULL (the caller wrote the pages): the kernel only zeroes the stale page tails
            const int64_t total = std::max<int64_t>(k_new ? (int64_t)m.n_tokens * c->shape.Hkv * (c->shape.D / 8) * 2 : 0,
                                                    (int64_t)m.n_reqs * 2 * c->shape.Hkv * (c->shape.B - 1) * (c->shape.D / 8));
            const int grid = (int)std::min<int64_t>((total + 255) / 256, (int64_t)c->n_sm * 8);
            kv_append_kernel<<<grid, 256, 0, stream>>>(m, c->shape, static_cast<const uint4*>(k_new),
                                                       static_cast<const uint4*>(v_new),
                                                       static_cast<__nv_bfloat16*>(kv_cache));
            CP_CUDA(cudaGetLastError());
            ++launches;
        }
        int rc;
#ifdef CP_DEBUG_VARIANTS
        if (!c->use_tc) {
            rc = c->shape.D == 128
                     ? launch_simt<128>(c, static_cast<const __nv_bfloat16*>(q), static_cast<const __nv_bfloat16*>(kv_cache),
                                        static_cast<__nv_bfloat16*>(out), stream)
                     : launch_simt<64>(c, static_cast<const __nv_bfloat16*>(q), static_cast<const __nv_bfloat16*>(kv_cache),
                                       static_cast<__nv_bfloat16*>(out), stream);
            launches += (m.n_work > 0) + (m.n_combine > 0);
            c->info.grid_attn = m.n_work;
            c->info.grid_combine = m.n_combine;
        } else
#endif
        {
            rc = launch_tc(c, static_cast<const __nv_bfloat16*>(q), kv_cache, static_cast<const float*>(kv_scale),
                           static_cast<__nv_bfloat16*>(out), stream, &launches, fused, k_new, v_new);
        }
        if (rc != CP_OK) return rc;
    }
    *launches_out = launches;
    return CP_OK;
}

// close a timed region [ts.start, stop recorded here]: the Table-1 features of the batch + which layer(s)
static int finish_timed(cp_ctx* c, TimedStep& ts, int32_t layer, int launches, cudaStream_t stream) {
    CP_CUDA(cudaEventRecord(ts.stop, stream));
    c->info.kernels_per_step = launches;
    cp_latency_row& row = ts.row;
    std::memcpy(row.feat, c->feat, sizeof(float) * 7);
    std::memcpy(row.feat + 7, c->mem_stats, sizeof(float) * 4);
    row.us = 0.f;
    row.n_prefill = c->n_prefill;
    row.n_decode = c->n_decode;
    row.layer = layer;
    row.iter = c->iter;
    ++c->ring_head;
    if (c->ring_head - c->ring_tail > kRing) c->ring_tail = c->ring_head - kRing;   // oldest rows overwritten
    return CP_OK;
}

static int attention_step(cp_ctx* c, int32_t layer, const void* q, const void* k_new, const void* v_new,
                          void* kv_cache, void* out, void* stream_, bool rope, void* kv_scale = nullptr) {
    if (!c) return CP_EINVAL;
    if (!c->have_batch) { cp_set_error("cp_attention_step: no batch built"); return CP_ESTATE; }
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    TimedStep& ts = c->ring[(size_t)(c->ring_head % kRing)];
    CP_CUDA(cudaEventRecord(ts.start, stream));
    int launches = 0;
    const int rc = issue_step(c, layer, q, k_new, v_new, kv_cache, out, stream, rope, kv_scale, &launches);
    if (rc != CP_OK) return rc;
    return finish_timed(c, ts, layer, launches, stream);
}

// One submission for all layers of an iteration (PAPER.md:201 counts kernel-launch latency among the fixed
// per-round overheads): the same kernels as n_layers cp_attention_step calls, ONE event pair, one latency row.
extern "C" int cp_attention_layers(cp_ctx* c, int32_t n_layers, const void* const* q, const void* const* k_new,
                                   const void* const* v_new, void* const* kv_cache, void* const* out, void* stream_) {
    if (!c || n_layers < 1 || !q || !kv_cache || !out || ((k_new == nullptr) != (v_new == nullptr))) {
        cp_set_error("cp_attention_layers: bad argument");
        return CP_EINVAL;
    }
    if (!c->have_batch) { cp_set_error("cp_attention_layers: no batch built"); return CP_ESTATE; }
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    TimedStep& ts = c->ring[(size_t)(c->ring_head % kRing)];
    CP_CUDA(cudaEventRecord(ts.start, stream));
    int total = 0;
    for (int32_t l = 0; l < n_layers; ++l) {
        int launches = 0;
        const int rc = issue_step(c, l, q[l], k_new ? k_new[l] : nullptr, v_new ? v_new[l] : nullptr, kv_cache[l], out[l],
                                  stream, false, nullptr, &launches);
        if (rc != CP_OK) return rc;
        total += launches;
    }
    return finish_timed(c, ts, -n_layers, total, stream);
}

extern "C" int cp_attention_step(cp_ctx* c, int32_t layer, const void* q, const void* k_new,
                                 const void* v_new, void* kv_cache, void* out, void* stream) {
    return attention_step(c, layer, q, k_new, v_new, kv_cache, out, stream, false);
}

extern "C" int cp_attention_step_fp8(cp_ctx* c, int32_t layer, const void* q, const void* k_new, const void* v_new,
                                     void* kv_cache8, void* kv_scale, void* out, void* stream) {
    if (!kv_scale || (reinterpret_cast<uintptr_t>(kv_scale) & 15)) { cp_set_error("cp_attention_step_fp8: kv_scale must be a 16-byte aligned device pointer"); return CP_EINVAL; }
    return attention_step(c, layer, q, k_new, v_new, kv_cache8, out, stream, false, kv_scale);
}

extern "C" int cp_attention_step_rope(cp_ctx* c, int32_t layer, const void* q, const void* k_new,
                                      const void* v_new, void* kv_cache, void* out, void* stream) {
    return attention_step(c, layer, q, k_new, v_new, kv_cache, out, stream, true);
}

// ------------------------------------------------------------------------------------
// H6: cp_latency_table
// ------------------------------------------------------------------------------------
extern "C" int cp_latency_table(cp_ctx* c, cp_latency_row* rows, int32_t cap, int32_t* n_out) {
    if (!c || !n_out || (cap > 0 && !rows) || cap < 0) { cp_set_error("cp_latency_table: bad argument"); return CP_EINVAL; }
    int32_t n = 0;
    while (c->ring_tail < c->ring_head && n < cap) {
        TimedStep& ts = c->ring[(size_t)(c->ring_tail % kRing)];
        CP_CUDA(cudaEventSynchronize(ts.stop));
        float ms = 0.f;
        CP_CUDA(cudaEventElapsedTime(&ms, ts.start, ts.stop));
        ts.row.us = ms * 1000.f;
        rows[n++] = ts.row;
        ++c->ring_tail;
    }
    *n_out = n;
    return CP_OK;
}

extern "C" int cp_set_memory_stats(cp_ctx* c, float used, float freemb, float allocated, float reserved) {
    if (!c) return CP_EINVAL;
    c->mem_stats[0] = used; c->mem_stats[1] = freemb; c->mem_stats[2] = allocated; c->mem_stats[3] = reserved;
    return CP_OK;
}

extern "C" int cp_get_batch_info(cp_ctx* c, cp_batch_info* info) {
    if (!c || !info) return CP_EINVAL;
    if (!c->have_batch) { cp_set_error("cp_get_batch_info: no batch built"); return CP_ESTATE; }
    *info = c->info;
    return CP_OK;
}
