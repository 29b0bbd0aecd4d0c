"""Reference scheduler -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Independent, step-by-step Python restatement of the paper's scheduler, in the
paper's order and notation.  libcp's C++ scheduler (cp_sched_*) must reproduce its
batch composition bit for bit; the two share no code.

  Aging priority        P_i = alpha (t - a_i) + beta r_i           Eq. 1
  chunk progress        r_i(n+1) = r_i(n) - c_i                    Eq. 2
  time-free key         K_i = -alpha a_i + beta r_i                Eq. 4
  max-heap on K, reinsertion after a chunk
  decode first, then rank prefills, requeue unfinished
  feasible bound        h_i = min(r_i, B_max - U_t)                Eq. 6
  token-budget chunk    c_i = h_i                                  Eq. 7
  candidate set         C_i = {1, h_i} U {k Delta}                 Eq. 8
  asymmetric score, argmin, tie -> larger c        Eq. 10-11, Alg. 1
  activity cap          C_t = min(C_max, S_max-|D_t|, floor((B_max-U_t)/L_min))
                                                                   Eq. 12
  minimum progress      m_i = min(r_i, L_min)                      Eq. 13
  APC decision (3 cases, tested in order)                          Eq. 14
  16 features (11 raw + 5 derived)                       Tables 1-2

Readings of silent/garbled points are those of SURVEY.md 8(c2) / DESIGN.md
("Scheduler readings" S1-S14).  PARITY WITH THE PAPER'S NUMBERS IS UNPINNED: the paper
prints no worked example and Tables 4-10 need ShareGPT, weights and the authors'
hardware.  Pinned by structure (tests/test_ref_scheduler.py): Eq. 3 order
equivalence, FCFS / shortest-remaining-first limits, closed-form overtake time,
conservation laws, Alg. 1 vs brute-force argmin and a closed form, Eq. 12-14 vs
exhaustive enumeration.

All arithmetic is IEEE fp64 in a fixed order (Python floats never contract to FMA).
"""
import heapq
import math

MODE_TOKEN_BUDGET = 0
MODE_LPRS = 1

PRED_LINEAR = 0
PRED_MLP = 1

N_FEAT = 16
FEATURE_NAMES = [
    "prefill_tokens", "decode_tokens", "batch_request_count",
    "sum_decode_context_len", "max_decode_context_len",
    "prefill_processed_tokens", "max_prefill_processed_tokens",
    "gpu_mem_used_mb", "gpu_mem_free_mb", "cuda_allocated_mb", "cuda_reserved_mb",
    "bias", "scheduled_tokens", "avg_decode_ctx", "decode_ctx_interaction",
    "prefill_interaction",
]


class SchedConfig:
    def __init__(self, alpha=100.0, beta=-1.0, B_max=2048, S_max=1024,
                 mode=MODE_TOKEN_BUDGET, apc=False, Delta=64, T_star=0.0,
                 lambda_u=1.0, lambda_o=2.0, C_max=4, L_min=64,
                 num_blocks=1 << 20, block_size=16, page_mb=0.0625,
                 pred_kind=PRED_LINEAR, pred_weights=None, feat_mu=None,
                 feat_inv_sigma=None):
        self.alpha = float(alpha)
        self.beta = float(beta)
        self.B_max = int(B_max)
        self.S_max = int(S_max)
        self.mode = int(mode)
        self.apc = bool(apc)
        self.Delta = int(Delta)
        self.T_star = float(T_star)
        self.lambda_u = float(lambda_u)
        self.lambda_o = float(lambda_o)
        self.C_max = int(C_max)
        self.L_min = int(L_min)
        self.num_blocks = int(num_blocks)
        self.block_size = int(block_size)
        self.page_mb = float(page_mb)
        self.pred_kind = int(pred_kind)
        # linear: 16 coefficients.  MLP: flat list W1[128][16], b1[128], W2[64][128],
        # b2[64], W3[32][64], b3[32], W4[1][32], b4[1] (row-major, out x in).
        self.pred_weights = [float(w) for w in (pred_weights or [0.0] * N_FEAT)]
        self.feat_mu = [float(x) for x in (feat_mu or [0.0] * N_FEAT)]
        self.feat_inv_sigma = [float(x) for x in (feat_inv_sigma or [1.0] * N_FEAT)]


MLP_DIMS = [16, 128, 64, 32, 1]


def mlp_num_weights():
    return sum(MLP_DIMS[i + 1] * MLP_DIMS[i] + MLP_DIMS[i + 1] for i in range(4))


class _Req:
    __slots__ = ("req_id", "arrival_us", "prompt_len", "output_len", "r",
                 "generated", "pages", "phase", "ttft_us", "finish_us")

    def __init__(self, req_id, arrival_us, prompt_len, output_len):
        self.req_id = req_id
        self.arrival_us = arrival_us
        self.prompt_len = prompt_len
        self.output_len = output_len
        self.r = prompt_len          # remaining prefill tokens r_i
        self.generated = 0
        self.pages = None
        self.phase = "future"        # future -> queued -> decode -> done
        self.ttft_us = -1
        self.finish_us = -1


class RefScheduler:
    def __init__(self, cfg: SchedConfig):
        self.cfg = cfg
        self.reqs = {}
        self.future = []             # min-heap on (arrival_us, req_id)
        self.heap = []               # max-heap on K: entries (-K, arrival_us, req_id)
        self.decoding = {}           # req_id -> _Req
        self.free_pages = list(range(cfg.num_blocks))   # already a valid min-heap
        self.used_pages = 0
        self.now_us = 0
        self.pending = None          # (decodes, prefills) of the formed iteration
        self.blocked_by_activity_cap = 0
        self.blocked_by_min_chunk = 0
        self.n_iters = 0

    # ---- Eq. 4 -----------------------------------------------------------------
    def key(self, rq):
        a = float(rq.arrival_us) * 1e-6
        return (-self.cfg.alpha * a) + (self.cfg.beta * float(rq.r))

    def _push(self, rq):
        heapq.heappush(self.heap, (-self.key(rq), rq.arrival_us, rq.req_id))

    def add_request(self, req_id, arrival_us, prompt_len, output_len):
        c = self.cfg
        if prompt_len < 1 or output_len < 1 or req_id in self.reqs:
            raise ValueError("bad request")
        need = (prompt_len + output_len + c.block_size - 1) // c.block_size
        if need > c.num_blocks:
            raise ValueError("request can never fit the pool")
        rq = _Req(int(req_id), int(arrival_us), int(prompt_len), int(output_len))
        self.reqs[rq.req_id] = rq
        heapq.heappush(self.future, (rq.arrival_us, rq.req_id))

    def next_arrival_us(self):
        return self.future[0][0] if self.future else -1

    def has_work(self):
        return bool(self.future or self.heap or self.decoding)

    # ---- predictor f_theta (Eq. 9); fixed summation order -------------------------
    def predict(self, x):
        c = self.cfg
        z = [(x[k] - c.feat_mu[k]) * c.feat_inv_sigma[k] for k in range(N_FEAT)]
        w = c.pred_weights
        if c.pred_kind == PRED_LINEAR:
            acc = 0.0
            for k in range(N_FEAT):
                acc = acc + w[k] * z[k]
            return acc
        pos = 0
        for li in range(4):
            n_in, n_out = MLP_DIMS[li], MLP_DIMS[li + 1]
            W = pos
            bpos = pos + n_out * n_in
            pos = bpos + n_out
            nz = []
            for o in range(n_out):
                acc = w[bpos + o]
                for i in range(n_in):
                    acc = acc + w[W + o * n_in + i] * z[i]
                if li < 3 and not (acc > 0.0):
                    acc = 0.0                     # ReLU (NaN -> 0)
                nz.append(acc)
            z = nz
        return z[0]

    # ---- Tables 1-2 -------------------------------------------------------------------
    def features(self, n_dec, sum_ctx, max_ctx, pf_tokens, n_pf, pf_proc, pf_proc_max):
        """16-dim vector for 'the batch if this candidate were accepted'."""
        c = self.cfg
        used = float(self.used_pages) * c.page_mb
        free = float(c.num_blocks - self.used_pages) * c.page_mb
        reserved = float(c.num_blocks) * c.page_mb
        prefill_tokens = float(pf_tokens)
        decode_tokens = float(n_dec)
        avg_ctx = float(sum_ctx) / float(max(n_dec, 1))
        return [
            prefill_tokens, decode_tokens, float(n_dec + n_pf),
            float(sum_ctx), float(max_ctx), float(pf_proc), float(pf_proc_max),
            used, free, used, reserved,
            1.0, decode_tokens + prefill_tokens, avg_ctx, decode_tokens * avg_ctx,
            prefill_tokens * float(pf_proc),
        ]

    # ---- Algorithm 1 (reconstructed; S10) -----------------
    def candidates(self, h):
        """Eq. 8, ascending."""
        C = {1, h}
        k = 1
        while k * self.cfg.Delta <= h:
            C.add(k * self.cfg.Delta)
            k += 1
        return sorted(C)

    def score(self, T_hat):
        c = self.cfg
        if T_hat <= c.T_star:
            return c.lambda_u * (c.T_star - T_hat)     # Eq. 10, underfill
        return c.lambda_o * (T_hat - c.T_star)         # Eq. 10, overflow

    def select_chunk(self, r_i, ctx_i, U_t, st):
        """st = (n_dec, sum_ctx, max_ctx, pf_tokens, n_pf, pf_proc, pf_proc_max)."""
        c = self.cfg
        h = min(r_i, c.B_max - U_t)
        if h <= 0:
            return 0
        n_dec, sum_ctx, max_ctx, pf_tokens, n_pf, pf_proc, pf_proc_max = st
        best = math.inf
        c_star = 0
        for cand in self.candidates(h):
            x = self.features(n_dec, sum_ctx, max_ctx, pf_tokens + cand, n_pf + 1,
                              pf_proc + ctx_i, max(pf_proc_max, ctx_i))
            sc = self.score(self.predict(x))
            if sc < best:
                best = sc
                c_star = cand
            elif sc == best and cand > c_star:          # tie -> larger c
                c_star = cand
        if c_star == 0 and U_t == 0 and h >= 1:         # starvation guard
            return 1
        return c_star

    # ---- APC ---------------------------------------------------------
    def activity_cap(self, n_dec, U_t):
        """Eq. 12, brackets read as floor (S9)."""
        c = self.cfg
        return min(c.C_max, c.S_max - n_dec, (c.B_max - U_t) // c.L_min)

    def apc_decision(self, c_star, r_i, h_i, P_size, C_t):
        """Eq. 13-14; the three cases are tested in the order printed."""
        m_i = min(r_i, self.cfg.L_min)                 # Eq. 13
        if P_size < C_t and c_star >= m_i:
            return c_star                              # accept
        if c_star < m_i and P_size == 0:
            return min(h_i, m_i)                       # warm start
        return 0                                       # block

    # ---- one scheduling round ---------------------------------------
    def next(self, now_us):
        """Form one iteration.  Returns [(req_id, q_len, ctx_off, [page ids])]:
        decodes first in (arrival_us, req_id) order, then prefill chunks in selection
        order.  Must be followed by commit() before the next call."""
        if self.pending is not None:
            raise RuntimeError("next() called twice without commit()")
        c = self.cfg
        self.now_us = int(now_us)
        # 1. arrivals enter the waiting heap
        while self.future and self.future[0][0] <= self.now_us:
            _, rid = heapq.heappop(self.future)
            rq = self.reqs[rid]
            rq.phase = "queued"
            self._push(rq)
        # 2. decode first
        dec = sorted(self.decoding.values(), key=lambda q: (q.arrival_us, q.req_id))
        dec = dec[: min(c.B_max, c.S_max)]
        U_t = len(dec)
        n_dec = len(dec)
        sum_ctx = 0
        max_ctx = 0
        for rq in dec:
            ctx = rq.prompt_len + rq.generated       # = ctx_off + 1 keys attended
            sum_ctx += ctx
            max_ctx = max(max_ctx, ctx)
        # 3. APC activity cap, evaluated once after decode admission (Eq. 12)
        C_t = self.activity_cap(n_dec, U_t) if c.apc else 0
        # 4. prefill selection loop
        chosen = []           # (rq, c_i)
        aside = []
        pf_tokens = 0
        pf_proc = 0
        pf_proc_max = 0
        while self.heap and U_t < c.B_max and n_dec + len(chosen) < c.S_max:
            if c.apc and len(chosen) >= 1 and len(chosen) >= C_t:
                break         # Eq. 14 would block every further candidate
            _, _, rid = heapq.heappop(self.heap)
            rq = self.reqs[rid]
            if rq.pages is None:                       # KV admission (S7)
                need = (rq.prompt_len + rq.output_len + c.block_size - 1) // c.block_size
                if need > len(self.free_pages):
                    aside.append(rq)
                    continue
            h_i = min(rq.r, c.B_max - U_t)             # Eq. 6
            ctx_i = rq.prompt_len - rq.r
            if c.mode == MODE_TOKEN_BUDGET:
                c_star = h_i                           # Eq. 7
            else:
                c_star = self.select_chunk(
                    rq.r, ctx_i, U_t,
                    (n_dec, sum_ctx, max_ctx, pf_tokens, len(chosen), pf_proc, pf_proc_max))
            if c.apc:
                c_i = self.apc_decision(c_star, rq.r, h_i, len(chosen), C_t)
                if c_i == 0:
                    if len(chosen) >= C_t:
                        self.blocked_by_activity_cap += 1
                    else:
                        self.blocked_by_min_chunk += 1
            else:
                c_i = c_star
            if c_i > 0:
                if rq.pages is None:
                    need = (rq.prompt_len + rq.output_len + c.block_size - 1) // c.block_size
                    rq.pages = [heapq.heappop(self.free_pages) for _ in range(need)]
                    self.used_pages += need
                chosen.append((rq, c_i))
                U_t += c_i
                pf_tokens += c_i
                pf_proc += ctx_i
                pf_proc_max = max(pf_proc_max, ctx_i)
            else:
                aside.append(rq)
        for rq in aside:                               # set aside: back, unchanged
            self._push(rq)
        self.pending = (dec, chosen) if (dec or chosen) else None   # empty: no commit
        out = [(rq.req_id, 1, rq.prompt_len + rq.generated - 1, list(rq.pages)) for rq in dec]
        out += [(rq.req_id, ci, rq.prompt_len - rq.r, list(rq.pages)) for rq, ci in chosen]
        return out

    def commit(self, iter_us):
        """Advance states after the iteration ran for iter_us microseconds."""
        if self.pending is None:
            raise RuntimeError("commit() without next()")
        dec, chosen = self.pending
        self.pending = None
        done_us = self.now_us + int(iter_us)
        self.n_iters += 1
        for rq in dec:
            rq.generated += 1
            if rq.generated >= rq.output_len:
                self._finish(rq, done_us)
        for rq, c_i in chosen:
            rq.r -= c_i                                # Eq. 2
            if rq.r > 0:
                self._push(rq)                         # reinsert with the new key
            else:
                rq.generated = 1                       # first token (S8)
                rq.ttft_us = done_us
                if rq.output_len == 1:
                    self._finish(rq, done_us)
                else:
                    rq.phase = "decode"
                    self.decoding[rq.req_id] = rq

    def _finish(self, rq, done_us):
        rq.phase = "done"
        rq.finish_us = done_us
        self.decoding.pop(rq.req_id, None)
        for p in rq.pages:
            heapq.heappush(self.free_pages, p)
        self.used_pages -= len(rq.pages)
        rq.pages = []


def pack_record(batch):
    """Canonical little-endian packing of one iteration's composition (for hashing)."""
    import struct
    b = bytearray()
    for req_id, q_len, ctx_off, pages in batch:
        b += struct.pack("<qiii", req_id, q_len, ctx_off, len(pages))
        b += struct.pack("<%di" % len(pages), *pages)
    return bytes(b)
