// cp_sched.cpp -- host-side scheduler of libcp (H0 in SURVEY.md 8(a)); no GPU code.
//
// Forms one chunked-prefill iteration per call, following arxiv/paper_2606_09061:
//   decode first, then prefills by aging key           PAPER.md:87, Eq. 4 (:99), :101
//   chunk = h_i (token budget, Eq. 6-7 :167-171) or Algorithm 1 (LPRS, :209-253)
//   Active Prefill Control gate                         Eq. 12-14 (:207, :261, :265)
// Compiled with -ffp-contract=off: every fp64 expression below is evaluated in the
// written order with no FMA contraction so that batch composition is bit-identical
// to the independent reference (oracle/ref_scheduler.py), which shares no code with
// this file.  Readings of points the paper leaves open: DESIGN.md S1-S14.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <limits>
#include <queue>
#include <unordered_map>
#include <vector>

#include "cp.h"

void cp_set_error(const char* fmt, ...);   // cp_api.cu / cp_error.cpp

namespace {

constexpr int kMlpDims[5] = {16, 128, 64, 32, 1};

enum class Phase : uint8_t { Future, Queued, Decode, Done };

struct Request {
    int64_t req_id = 0, arrival_us = 0;
    int32_t prompt_len = 0, output_len = 0;
    int32_t remaining = 0;      // r_i
    int32_t generated = 0;
    bool has_pages = false;
    Phase phase = Phase::Future;
    int64_t ttft_us = -1, finish_us = -1;
    std::vector<int32_t> pages;
};

struct WaitEntry {              // max-heap on K; ties: earlier arrival, smaller id
    double K;
    int64_t arrival_us, req_id;
    int32_t slot;
};
struct WaitLess {
    bool operator()(const WaitEntry& a, const WaitEntry& b) const {
        if (a.K != b.K) return a.K < b.K;
        if (a.arrival_us != b.arrival_us) return a.arrival_us > b.arrival_us;
        return a.req_id > b.req_id;
    }
};
struct FutureEntry { int64_t arrival_us, req_id; int32_t slot; };
struct FutureGreater {
    bool operator()(const FutureEntry& a, const FutureEntry& b) const {
        if (a.arrival_us != b.arrival_us) return a.arrival_us > b.arrival_us;
        return a.req_id > b.req_id;
    }
};

struct BatchState {             // what Tables 1-2 need about the batch formed so far
    int32_t n_dec = 0;
    int64_t sum_ctx = 0;
    int32_t max_ctx = 0;
    int32_t pf_tokens = 0;
    int32_t n_pf = 0;
    int64_t pf_proc = 0;
    int32_t pf_proc_max = 0;
};

}  // namespace

struct cp_sched {
    cp_sched_config cfg{};
    std::vector<double> w, mu, inv_sigma;
    std::vector<Request> reqs;
    std::unordered_map<int64_t, int32_t> slot_of;
    std::priority_queue<FutureEntry, std::vector<FutureEntry>, FutureGreater> future;
    std::priority_queue<WaitEntry, std::vector<WaitEntry>, WaitLess> waiting;
    std::vector<int32_t> decoding;                    // slots in decode phase
    std::priority_queue<int32_t, std::vector<int32_t>, std::greater<int32_t>> free_pages;
    int64_t used_pages = 0;
    int64_t now_us = 0;
    bool pending = false;
    std::vector<int32_t> pend_dec;                    // slots
    std::vector<std::pair<int32_t, int32_t>> pend_pf; // (slot, c_i)
    int64_t n_iters = 0, blocked_cap = 0, blocked_min = 0;

    double key(const Request& r) const {              // Eq. 4
        double a = static_cast<double>(r.arrival_us) * 1e-6;
        double t1 = -cfg.alpha * a;
        double t2 = cfg.beta * static_cast<double>(r.remaining);
        return t1 + t2;
    }
    void push_waiting(int32_t slot) {
        const Request& r = reqs[slot];
        waiting.push(WaitEntry{key(r), r.arrival_us, r.req_id, slot});
    }
    int32_t pages_needed(const Request& r) const {
        return (r.prompt_len + r.output_len + cfg.block_size - 1) / cfg.block_size;
    }

    // Tables 1-2: the batch "if this candidate were accepted"
    void features(const BatchState& b, double* x) const {
        double used = static_cast<double>(used_pages) * cfg.page_mb;
        double freemb = static_cast<double>(cfg.num_blocks - used_pages) * cfg.page_mb;
        double reserved = static_cast<double>(cfg.num_blocks) * cfg.page_mb;
        double prefill_tokens = static_cast<double>(b.pf_tokens);
        double decode_tokens = static_cast<double>(b.n_dec);
        double avg_ctx = static_cast<double>(b.sum_ctx) /
                         static_cast<double>(std::max(b.n_dec, 1));
        x[0] = prefill_tokens;
        x[1] = decode_tokens;
        x[2] = static_cast<double>(b.n_dec + b.n_pf);
        x[3] = static_cast<double>(b.sum_ctx);
        x[4] = static_cast<double>(b.max_ctx);
        x[5] = static_cast<double>(b.pf_proc);
        x[6] = static_cast<double>(b.pf_proc_max);
        x[7] = used;
        x[8] = freemb;
        x[9] = used;
        x[10] = reserved;
        x[11] = 1.0;
        x[12] = decode_tokens + prefill_tokens;
        x[13] = avg_ctx;
        x[14] = decode_tokens * avg_ctx;
        x[15] = prefill_tokens * static_cast<double>(b.pf_proc);
    }

    double predict(const double* x) const {           // Eq. 9, fixed summation order
        double z[128], nz[128];
        for (int k = 0; k < 16; ++k) {
            double d = x[k] - mu[k];
            z[k] = d * inv_sigma[k];
        }
        if (cfg.pred_kind == CP_PRED_LINEAR) {
            double acc = 0.0;
            for (int k = 0; k < 16; ++k) {
                double p = w[k] * z[k];
                acc = acc + p;
            }
            return acc;
        }
        size_t pos = 0;
        for (int li = 0; li < 4; ++li) {
            const int n_in = kMlpDims[li], n_out = kMlpDims[li + 1];
            const double* W = w.data() + pos;
            const double* bias = W + static_cast<size_t>(n_out) * n_in;
            pos += static_cast<size_t>(n_out) * n_in + n_out;
            for (int o = 0; o < n_out; ++o) {
                double acc = bias[o];
                for (int i = 0; i < n_in; ++i) {
                    double p = W[o * n_in + i] * z[i];
                    acc = acc + p;
                }
                if (li < 3 && !(acc > 0.0)) acc = 0.0;
                nz[o] = acc;
            }
            std::memcpy(z, nz, sizeof(double) * n_out);
        }
        return z[0];
    }

    double score(double t_hat) const {                // Eq. 10
        if (t_hat <= cfg.T_star) return cfg.lambda_u * (cfg.T_star - t_hat);
        return cfg.lambda_o * (t_hat - cfg.T_star);
    }

    // Algorithm 1
    int32_t select_chunk(int32_t r_i, int32_t ctx_i, int32_t U_t, const BatchState& b) const {
        int32_t h = std::min(r_i, cfg.B_max - U_t);
        if (h <= 0) return 0;
        std::vector<int32_t> cands;                   // Eq. 8
        cands.push_back(1);
        for (int64_t k = cfg.Delta; k <= h; k += cfg.Delta) cands.push_back(static_cast<int32_t>(k));
        cands.push_back(h);
        std::sort(cands.begin(), cands.end());
        cands.erase(std::unique(cands.begin(), cands.end()), cands.end());
        double best = std::numeric_limits<double>::infinity();
        int32_t c_star = 0;
        BatchState t = b;
        t.n_pf = b.n_pf + 1;
        t.pf_proc = b.pf_proc + ctx_i;
        t.pf_proc_max = std::max(b.pf_proc_max, ctx_i);
        double x[16];
        for (int32_t c : cands) {
            t.pf_tokens = b.pf_tokens + c;
            features(t, x);
            double sc = score(predict(x));
            if (sc < best) { best = sc; c_star = c; }
            else if (sc == best && c > c_star) { c_star = c; }     // tie -> larger c
        }
        if (c_star == 0 && U_t == 0 && h >= 1) return 1;           // starvation guard
        return c_star;
    }

    int32_t activity_cap(int32_t n_dec, int32_t U_t) const {       // Eq. 12 (floor)
        int32_t by_budget = (cfg.B_max - U_t) / cfg.L_min;         // operands >= 0
        return std::min(cfg.C_max, std::min(cfg.S_max - n_dec, by_budget));
    }
    int32_t apc_decision(int32_t c_star, int32_t r_i, int32_t h_i, int32_t P, int32_t C_t) const {
        int32_t m_i = std::min(r_i, cfg.L_min);                    // Eq. 13
        if (P < C_t && c_star >= m_i) return c_star;               // Eq. 14, in order
        if (c_star < m_i && P == 0) return std::min(h_i, m_i);
        return 0;
    }

    void finish(int32_t slot, int64_t done_us) {
        Request& r = reqs[slot];
        r.phase = Phase::Done;
        r.finish_us = done_us;
        auto it = std::find(decoding.begin(), decoding.end(), slot);
        if (it != decoding.end()) decoding.erase(it);
        for (int32_t p : r.pages) free_pages.push(p);
        used_pages -= static_cast<int64_t>(r.pages.size());
        r.pages.clear();
        r.pages.shrink_to_fit();
    }
};

// ------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------
extern "C" {

int cp_sched_create(const cp_sched_config* cfg, cp_sched** out) {
    if (!cfg || !out) { cp_set_error("cp_sched_create: null argument"); return CP_EINVAL; }
    if (cfg->B_max < 1 || cfg->S_max < 1 || cfg->block_size < 1 || cfg->num_blocks < 1 ||
        cfg->Delta < 1 || cfg->L_min < 1 || cfg->num_blocks > INT32_MAX) {
        cp_set_error("cp_sched_create: bad limits");
        return CP_EINVAL;
    }
    // Eq. 12 with C_max < 1 or L_min > B_max gives C_t = 0 on an empty batch: literal Eq. 14 then blocks every
    // candidate for ever (no round could start a prefill) -- a configuration error, not a schedule
    if (cfg->apc && (cfg->C_max < 1 || cfg->L_min > cfg->B_max)) {
        cp_set_error("cp_sched_create: APC needs C_max >= 1 and L_min <= B_max");
        return CP_EINVAL;
    }
    if (cfg->mode == CP_MODE_LPRS && !(cfg->lambda_u >= 0.0 && cfg->lambda_o >= 0.0)) {
        cp_set_error("cp_sched_create: lambda_u, lambda_o must be >= 0 (Eq. 10; the paper takes lambda_o > lambda_u)");
        return CP_EINVAL;
    }
    size_t need = 16;
    if (cfg->pred_kind == CP_PRED_MLP) {
        need = 0;
        for (int i = 0; i < 4; ++i) need += static_cast<size_t>(kMlpDims[i + 1]) * kMlpDims[i] + kMlpDims[i + 1];
    } else if (cfg->pred_kind != CP_PRED_LINEAR) {
        cp_set_error("cp_sched_create: unknown predictor kind");
        return CP_EINVAL;
    }
    if (cfg->mode != CP_MODE_TOKEN_BUDGET && cfg->mode != CP_MODE_LPRS) {
        cp_set_error("cp_sched_create: unknown mode");
        return CP_EINVAL;
    }
    cp_sched* s = new cp_sched();
    s->cfg = *cfg;
    s->w.assign(need, 0.0);
    if (cfg->pred_weights) {
        if (static_cast<size_t>(cfg->n_pred_weights) != need) {
            delete s;
            cp_set_error("cp_sched_create: expected %zu predictor weights, got %d", need,
                         cfg->n_pred_weights);
            return CP_EINVAL;
        }
        std::copy(cfg->pred_weights, cfg->pred_weights + need, s->w.begin());
    }
    s->mu.assign(16, 0.0);
    s->inv_sigma.assign(16, 1.0);
    if (cfg->feat_mu) std::copy(cfg->feat_mu, cfg->feat_mu + 16, s->mu.begin());
    if (cfg->feat_inv_sigma) std::copy(cfg->feat_inv_sigma, cfg->feat_inv_sigma + 16, s->inv_sigma.begin());
    s->cfg.pred_weights = nullptr;
    s->cfg.feat_mu = nullptr;
    s->cfg.feat_inv_sigma = nullptr;
    {   // lowest free page id first (S7)
        std::vector<int32_t> ids(static_cast<size_t>(cfg->num_blocks));
        for (size_t i = 0; i < ids.size(); ++i) ids[i] = static_cast<int32_t>(i);
        s->free_pages = decltype(s->free_pages)(std::greater<int32_t>(), std::move(ids));
    }
    *out = s;
    return CP_OK;
}

int cp_sched_destroy(cp_sched* s) {
    delete s;
    return CP_OK;
}

int cp_sched_add_request(cp_sched* s, int64_t req_id, int64_t arrival_us, int32_t prompt_len,
                         int32_t output_len) {
    if (!s) return CP_EINVAL;
    if (prompt_len < 1 || output_len < 1 || s->slot_of.count(req_id)) {
        cp_set_error("cp_sched_add_request: bad request %lld", (long long)req_id);
        return CP_EINVAL;
    }
    Request r;
    r.req_id = req_id;
    r.arrival_us = arrival_us;
    r.prompt_len = prompt_len;
    r.output_len = output_len;
    r.remaining = prompt_len;
    if (s->pages_needed(r) > s->cfg.num_blocks) {
        cp_set_error("cp_sched_add_request: request %lld can never fit the pool", (long long)req_id);
        return CP_ECAPACITY;
    }
    int32_t slot = static_cast<int32_t>(s->reqs.size());
    s->reqs.push_back(std::move(r));
    s->slot_of[req_id] = slot;
    s->future.push(FutureEntry{arrival_us, req_id, slot});
    return CP_OK;
}

int cp_sched_next(cp_sched* s, int64_t now_us, cp_req_desc* out, int32_t cap, int32_t* n_out) {
    if (!s || !out || !n_out) return CP_EINVAL;
    if (s->pending) { cp_set_error("cp_sched_next: previous iteration not committed"); return CP_ESTATE; }
    const cp_sched_config& c = s->cfg;
    s->now_us = now_us;
    // 1. arrivals
    while (!s->future.empty() && s->future.top().arrival_us <= now_us) {
        int32_t slot = s->future.top().slot;
        s->future.pop();
        s->reqs[slot].phase = Phase::Queued;
        s->push_waiting(slot);
    }
    // 2. decode first, (arrival_us, req_id) order, truncated to min(B_max, S_max)
    std::vector<int32_t> dec = s->decoding;
    std::sort(dec.begin(), dec.end(), [&](int32_t a, int32_t b) {
        const Request& ra = s->reqs[a];
        const Request& rb = s->reqs[b];
        if (ra.arrival_us != rb.arrival_us) return ra.arrival_us < rb.arrival_us;
        return ra.req_id < rb.req_id;
    });
    size_t lim = static_cast<size_t>(std::min(c.B_max, c.S_max));
    if (dec.size() > lim) dec.resize(lim);
    BatchState b;
    b.n_dec = static_cast<int32_t>(dec.size());
    int32_t U_t = b.n_dec;
    for (int32_t slot : dec) {
        const Request& r = s->reqs[slot];
        int32_t ctx = r.prompt_len + r.generated;
        b.sum_ctx += ctx;
        b.max_ctx = std::max(b.max_ctx, ctx);
    }
    // 3. activity cap, once, after decode admission
    const int32_t C_t = c.apc ? s->activity_cap(b.n_dec, U_t) : 0;
    // 4. prefill selection
    std::vector<std::pair<int32_t, int32_t>> chosen;
    std::vector<int32_t> aside;
    while (!s->waiting.empty() && U_t < c.B_max &&
           b.n_dec + static_cast<int32_t>(chosen.size()) < c.S_max) {
        const int32_t P = static_cast<int32_t>(chosen.size());
        if (c.apc && P >= 1 && P >= C_t) break;
        int32_t slot = s->waiting.top().slot;
        s->waiting.pop();
        Request& r = s->reqs[slot];
        if (!r.has_pages && static_cast<size_t>(s->pages_needed(r)) > s->free_pages.size()) {
            aside.push_back(slot);
            continue;
        }
        const int32_t h_i = std::min(r.remaining, c.B_max - U_t);      // Eq. 6
        const int32_t ctx_i = r.prompt_len - r.remaining;
        int32_t c_star;
        if (c.mode == CP_MODE_TOKEN_BUDGET) c_star = h_i;              // Eq. 7
        else c_star = s->select_chunk(r.remaining, ctx_i, U_t, b);
        int32_t c_i = c_star;
        if (c.apc) {
            c_i = s->apc_decision(c_star, r.remaining, h_i, P, C_t);
            if (c_i == 0) { if (P >= C_t) ++s->blocked_cap; else ++s->blocked_min; }
        }
        if (c_i > 0) {
            if (!r.has_pages) {
                int32_t need = s->pages_needed(r);
                r.pages.reserve(need);
                for (int32_t k = 0; k < need; ++k) { r.pages.push_back(s->free_pages.top()); s->free_pages.pop(); }
                s->used_pages += need;
                r.has_pages = true;
            }
            chosen.emplace_back(slot, c_i);
            U_t += c_i;
            b.pf_tokens += c_i;
            b.n_pf += 1;
            b.pf_proc += ctx_i;
            b.pf_proc_max = std::max(b.pf_proc_max, ctx_i);
        } else {
            aside.push_back(slot);
        }
    }
    for (int32_t slot : aside) s->push_waiting(slot);
    const size_t n = dec.size() + chosen.size();
    if (n > static_cast<size_t>(cap)) {
        // undo nothing: the formed batch is kept pending so the caller can retry? No --
        // keep it simple and deterministic: this is a caller bug.
        for (auto& pc : chosen) s->push_waiting(pc.first);
        cp_set_error("cp_sched_next: cap %d too small for %zu requests", cap, n);
        return CP_ECAPACITY;
    }
    size_t k = 0;
    for (int32_t slot : dec) {
        const Request& r = s->reqs[slot];
        out[k++] = cp_req_desc{r.req_id, 1, r.prompt_len + r.generated - 1, r.pages.data(),
                               static_cast<int32_t>(r.pages.size()), 0};
    }
    for (auto& pc : chosen) {
        const Request& r = s->reqs[pc.first];
        out[k++] = cp_req_desc{r.req_id, pc.second, r.prompt_len - r.remaining, r.pages.data(),
                               static_cast<int32_t>(r.pages.size()), CP_REQ_PREFILL};
    }
    *n_out = static_cast<int32_t>(n);
    s->pending = n > 0;
    s->pend_dec = std::move(dec);
    s->pend_pf = std::move(chosen);
    return CP_OK;
}

int cp_sched_commit(cp_sched* s, int64_t iter_us) {
    if (!s) return CP_EINVAL;
    if (!s->pending) { cp_set_error("cp_sched_commit: nothing to commit"); return CP_ESTATE; }
    s->pending = false;
    const int64_t done_us = s->now_us + iter_us;
    ++s->n_iters;
    for (int32_t slot : s->pend_dec) {
        Request& r = s->reqs[slot];
        r.generated += 1;
        if (r.generated >= r.output_len) s->finish(slot, done_us);
    }
    for (auto& pc : s->pend_pf) {
        Request& r = s->reqs[pc.first];
        r.remaining -= pc.second;                                      // Eq. 2
        if (r.remaining > 0) {
            s->push_waiting(pc.first);
        } else {
            r.generated = 1;
            r.ttft_us = done_us;
            if (r.output_len == 1) s->finish(pc.first, done_us);
            else { r.phase = Phase::Decode; s->decoding.push_back(pc.first); }
        }
    }
    s->pend_dec.clear();
    s->pend_pf.clear();
    return CP_OK;
}

int cp_sched_next_arrival(cp_sched* s, int64_t* arrival_us) {
    if (!s || !arrival_us) return CP_EINVAL;
    *arrival_us = s->future.empty() ? -1 : s->future.top().arrival_us;
    return CP_OK;
}

int cp_sched_has_work(cp_sched* s, int32_t* has_work) {
    if (!s || !has_work) return CP_EINVAL;
    *has_work = !(s->future.empty() && s->waiting.empty() && s->decoding.empty());
    return CP_OK;
}

int cp_sched_get_stats(cp_sched* s, cp_sched_stats* st) {
    if (!s || !st) return CP_EINVAL;
    st->n_iters = s->n_iters;
    st->blocked_by_activity_cap = s->blocked_cap;
    st->blocked_by_min_chunk = s->blocked_min;
    st->used_pages = s->used_pages;
    st->n_waiting = static_cast<int32_t>(s->waiting.size());
    st->n_decoding = static_cast<int32_t>(s->decoding.size());
    st->n_future = static_cast<int32_t>(s->future.size());
    return CP_OK;
}

int cp_sched_request_times(cp_sched* s, int64_t req_id, int64_t* ttft_us, int64_t* finish_us) {
    if (!s) return CP_EINVAL;
    auto it = s->slot_of.find(req_id);
    if (it == s->slot_of.end()) { cp_set_error("unknown request"); return CP_EINVAL; }
    if (ttft_us) *ttft_us = s->reqs[it->second].ttft_us;
    if (finish_us) *finish_us = s->reqs[it->second].finish_us;
    return CP_OK;
}

int cp_sched_predict(cp_sched* s, const double* x16, double* t_hat) {
    if (!s || !x16 || !t_hat) return CP_EINVAL;
    *t_hat = s->predict(x16);
    return CP_OK;
}

int cp_sched_select_chunk(cp_sched* s, int32_t r_i, int32_t ctx_i, int32_t U_t, int32_t n_dec,
                          int64_t sum_ctx, int32_t max_ctx, int32_t pf_tokens, int32_t n_pf,
                          int64_t pf_proc, int32_t pf_proc_max, int32_t* c_star) {
    if (!s || !c_star) return CP_EINVAL;
    BatchState b;
    b.n_dec = n_dec; b.sum_ctx = sum_ctx; b.max_ctx = max_ctx; b.pf_tokens = pf_tokens;
    b.n_pf = n_pf; b.pf_proc = pf_proc; b.pf_proc_max = pf_proc_max;
    *c_star = s->select_chunk(r_i, ctx_i, U_t, b);
    return CP_OK;
}

}  // extern "C"
