"""Thin ctypes binding over the C ABI of include/cp.h (argument marshalling only).

Every step of the hot path runs inside libcp.so; PyTorch appears here only as the
owner of device memory and streams (tensors are passed as raw data_ptr()).  There is
no CPU fallback: load() raises if libcp.so is missing or lacks a symbol.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcp.so")

CP_OK, CP_EINVAL, CP_ECAPACITY, CP_ECUDA, CP_ESTATE = 0, -1, -2, -3, -4
CP_REQ_PREFILL = 1
CP_KV_BF16, CP_KV_E4M3 = 0, 1
CP_MODE_TOKEN_BUDGET, CP_MODE_LPRS = 0, 1
CP_PRED_LINEAR, CP_PRED_MLP = 0, 1
CP_NUM_RAW_FEATURES = 11

EXPORTS = [
    "cp_last_error", "cp_create", "cp_destroy", "cp_build_batch", "cp_attention_step",
    "cp_latency_table", "cp_set_memory_stats", "cp_get_batch_info", "cp_sched_create",
    "cp_sched_destroy", "cp_sched_add_request", "cp_sched_next", "cp_sched_commit",
    "cp_sched_next_arrival", "cp_sched_has_work", "cp_sched_get_stats",
    "cp_sched_request_times", "cp_sched_predict", "cp_sched_select_chunk",
    "cp_enable_rope", "cp_attention_step_rope", "cp_attention_step_fp8", "cp_attention_layers",
    "cp_decode_attention_static",
]


class cp_config(C.Structure):
    _fields_ = [("num_q_heads", C.c_int32), ("num_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("block_size", C.c_int32), ("num_layers", C.c_int32), ("num_blocks", C.c_int64),
                ("sm_scale", C.c_float), ("max_tokens", C.c_int32), ("max_reqs", C.c_int32),
                ("max_total_pages", C.c_int64), ("max_partial_rows", C.c_int64),
                ("device", C.c_int32), ("kernel_variant", C.c_int32), ("kv_dtype", C.c_int32),
                ("reserved", C.c_int32), ("max_scratch_pages", C.c_int64)]


class cp_req_desc(C.Structure):
    _fields_ = [("req_id", C.c_int64), ("q_len", C.c_int32), ("ctx_off", C.c_int32),
                ("block_table", C.POINTER(C.c_int32)), ("n_blocks", C.c_int32), ("flags", C.c_int32)]


class cp_latency_row(C.Structure):
    _fields_ = [("feat", C.c_float * CP_NUM_RAW_FEATURES), ("us", C.c_float),
                ("n_prefill", C.c_int32), ("n_decode", C.c_int32), ("layer", C.c_int32),
                ("iter", C.c_int64)]


class cp_batch_info(C.Structure):
    _fields_ = [("n_reqs", C.c_int32), ("n_tokens", C.c_int32), ("n_work_items", C.c_int32),
                ("n_combine_items", C.c_int32), ("n_tc_items", C.c_int32),
                ("n_partial_rows", C.c_int64), ("kernels_per_step", C.c_int32),
                ("grid_attn", C.c_int32), ("grid_combine", C.c_int32), ("alg_flops", C.c_double),
                ("alg_bytes", C.c_double), ("split", C.c_int32)]


class cp_sched_config(C.Structure):
    _fields_ = [("alpha", C.c_double), ("beta", C.c_double), ("B_max", C.c_int32),
                ("S_max", C.c_int32), ("mode", C.c_int32), ("apc", C.c_int32),
                ("Delta", C.c_int32), ("C_max", C.c_int32), ("L_min", C.c_int32),
                ("block_size", C.c_int32), ("num_blocks", C.c_int64), ("T_star", C.c_double),
                ("lambda_u", C.c_double), ("lambda_o", C.c_double), ("page_mb", C.c_double),
                ("pred_kind", C.c_int32), ("n_pred_weights", C.c_int32),
                ("pred_weights", C.POINTER(C.c_double)), ("feat_mu", C.POINTER(C.c_double)),
                ("feat_inv_sigma", C.POINTER(C.c_double))]


class cp_sched_stats(C.Structure):
    _fields_ = [("n_iters", C.c_int64), ("blocked_by_activity_cap", C.c_int64),
                ("blocked_by_min_chunk", C.c_int64), ("used_pages", C.c_int64),
                ("n_waiting", C.c_int32), ("n_decoding", C.c_int32), ("n_future", C.c_int32)]


class CpError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libcp error {code}: {msg}")
        self.code = code


_lib = None


def load(path: Optional[str] = None):
    """dlopen libcp.so and check that every symbol of include/cp.h is exported."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise ImportError(f"{p} is missing: build it with `python -m paper_2606_09061_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(p)
    for name in EXPORTS:
        if not hasattr(lib, name):
            raise ImportError(f"{p} does not export {name}")
    lib.cp_last_error.restype = C.c_char_p
    for name in EXPORTS[1:]:
        getattr(lib, name).restype = C.c_int
    lib.cp_create.argtypes = [C.POINTER(cp_config), C.POINTER(C.c_void_p)]
    lib.cp_destroy.argtypes = [C.c_void_p]
    lib.cp_build_batch.argtypes = [C.c_void_p, C.POINTER(cp_req_desc), C.c_int32, C.c_void_p]
    lib.cp_attention_step.argtypes = [C.c_void_p, C.c_int32] + [C.c_void_p] * 6
    lib.cp_attention_step_rope.argtypes = [C.c_void_p, C.c_int32] + [C.c_void_p] * 6
    lib.cp_attention_step_fp8.argtypes = [C.c_void_p, C.c_int32] + [C.c_void_p] * 7
    lib.cp_attention_layers.argtypes = [C.c_void_p, C.c_int32] + [C.POINTER(C.c_void_p)] * 5 + [C.c_void_p]
    lib.cp_enable_rope.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
    lib.cp_latency_table.argtypes = [C.c_void_p, C.POINTER(cp_latency_row), C.c_int32,
                                     C.POINTER(C.c_int32)]
    lib.cp_set_memory_stats.argtypes = [C.c_void_p] + [C.c_float] * 4
    lib.cp_get_batch_info.argtypes = [C.c_void_p, C.POINTER(cp_batch_info)]
    lib.cp_sched_create.argtypes = [C.POINTER(cp_sched_config), C.POINTER(C.c_void_p)]
    lib.cp_sched_destroy.argtypes = [C.c_void_p]
    lib.cp_sched_add_request.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_int32, C.c_int32]
    lib.cp_sched_next.argtypes = [C.c_void_p, C.c_int64, C.POINTER(cp_req_desc), C.c_int32,
                                  C.POINTER(C.c_int32)]
    lib.cp_sched_commit.argtypes = [C.c_void_p, C.c_int64]
    lib.cp_sched_next_arrival.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
    lib.cp_sched_has_work.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
    lib.cp_sched_get_stats.argtypes = [C.c_void_p, C.POINTER(cp_sched_stats)]
    lib.cp_sched_request_times.argtypes = [C.c_void_p, C.c_int64, C.POINTER(C.c_int64),
                                           C.POINTER(C.c_int64)]
    lib.cp_sched_predict.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.cp_sched_select_chunk.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32,
                                          C.c_int64, C.c_int32, C.c_int32, C.c_int32, C.c_int64,
                                          C.c_int32, C.POINTER(C.c_int32)]
    lib.cp_decode_attention_static.argtypes = [C.c_void_p] * 4 + [C.c_int32] * 6 + [C.c_float, C.c_int32, C.c_void_p, C.c_void_p]
    if path is None:
        _lib = lib
    return lib


def _check(rc: int):
    if rc != CP_OK:
        raise CpError(rc, load().cp_last_error().decode(errors="replace"))


def make_descs(q_len: Sequence[int], ctx_off: Sequence[int], block_tables: Sequence[np.ndarray],
               req_ids: Optional[Sequence[int]] = None, flags: Optional[Sequence[int]] = None):
    """Marshal a batch into a cp_req_desc array (keeps the int32 tables alive)."""
    n = len(q_len)
    arr = (cp_req_desc * max(n, 1))()
    keep = []
    for j in range(n):
        bt = np.ascontiguousarray(block_tables[j], dtype=np.int32)
        keep.append(bt)
        arr[j].req_id = int(req_ids[j]) if req_ids is not None else j
        arr[j].q_len = int(q_len[j])
        arr[j].ctx_off = int(ctx_off[j])
        arr[j].block_table = bt.ctypes.data_as(C.POINTER(C.c_int32))
        arr[j].n_blocks = len(bt)
        arr[j].flags = int(flags[j]) if flags is not None else 0
    return arr, keep


def rope_inv_freq(head_dim: int, theta: float = 10000.0) -> np.ndarray:
    """The usual rotary frequencies w_f = theta^(-2f/D), float64 [D/2] (argument of cp_enable_rope)."""
    return np.float64(theta) ** (-np.arange(0, head_dim, 2, dtype=np.float64) / head_dim)


def _ptr(t) -> Optional[int]:
    if t is None:
        return None
    return int(t.data_ptr()) if hasattr(t, "data_ptr") else int(t)


CP_STATIC_MAX_PARTIAL_ROWS = 4096


def cp_decode_attention_static(q, kv_cache, block_tables, kv_len, n_reqs, max_pages_per_req, num_q_heads,
                               num_kv_heads, head_dim, block_size, sm_scale, n_splits, out, stream=None):
    """The no-allocation entry point (include/cp.h): device pointers / tensors in, two kernels enqueued, no context."""
    _check(load().cp_decode_attention_static(_ptr(q), _ptr(kv_cache), _ptr(block_tables), _ptr(kv_len), n_reqs,
                                             max_pages_per_req, num_q_heads, num_kv_heads, head_dim, block_size,
                                             float(sm_scale), n_splits, _ptr(out), _ptr(stream)))


class Context:
    """cp_create / cp_build_batch / cp_attention_step / cp_latency_table, same names."""

    def __init__(self, num_q_heads, num_kv_heads, head_dim, num_blocks, block_size=16,
                 num_layers=1, sm_scale=None, max_tokens=8192, max_reqs=1024,
                 max_total_pages=None, max_partial_rows=0, device=0, kernel_variant=0, kv_dtype=0,
                 max_scratch_pages=0):
        self.lib = load()
        if sm_scale is None:
            sm_scale = float(np.float32(1.0) / np.sqrt(np.float32(head_dim)))
        if max_total_pages is None:
            max_total_pages = int(num_blocks)
        self.cfg = cp_config(num_q_heads, num_kv_heads, head_dim, block_size, num_layers,
                             num_blocks, sm_scale, max_tokens, max_reqs, max_total_pages,
                             max_partial_rows, device, kernel_variant, kv_dtype, 0, max_scratch_pages)
        self.handle = C.c_void_p()
        _check(self.lib.cp_create(C.byref(self.cfg), C.byref(self.handle)))
        self._keep = None

    def cp_build_batch(self, q_len=None, ctx_off=None, block_tables=None, stream=None,
                       descs=None, n=None, flags=None):
        if descs is None:
            descs, self._keep = make_descs(q_len, ctx_off, block_tables, flags=flags)
            n = len(q_len)
        _check(self.lib.cp_build_batch(self.handle, descs, n, _ptr(stream)))

    def cp_attention_step(self, layer, q, k_new, v_new, kv_cache, out, stream=None):
        _check(self.lib.cp_attention_step(self.handle, layer, _ptr(q), _ptr(k_new), _ptr(v_new),
                                          _ptr(kv_cache), _ptr(out), _ptr(stream)))

    def cp_enable_rope(self, inv_freq):
        f = np.ascontiguousarray(inv_freq, dtype=np.float64)
        if f.shape != (self.cfg.head_dim // 2,):
            raise ValueError(f"inv_freq must have head_dim/2 = {self.cfg.head_dim // 2} entries")
        _check(self.lib.cp_enable_rope(self.handle, f.ctypes.data_as(C.POINTER(C.c_double))))

    def cp_attention_step_rope(self, layer, q, k_new, v_new, kv_cache, out, stream=None):
        _check(self.lib.cp_attention_step_rope(self.handle, layer, _ptr(q), _ptr(k_new), _ptr(v_new),
                                               _ptr(kv_cache), _ptr(out), _ptr(stream)))

    def cp_attention_step_fp8(self, layer, q, k_new, v_new, kv_cache8, kv_scale, out, stream=None):
        _check(self.lib.cp_attention_step_fp8(self.handle, layer, _ptr(q), _ptr(k_new), _ptr(v_new),
                                              _ptr(kv_cache8), _ptr(kv_scale), _ptr(out), _ptr(stream)))

    @staticmethod
    def pointer_array(ptrs):
        """HOST array of device pointers for cp_attention_layers (build once, reuse every iteration)."""
        return (C.c_void_p * len(ptrs))(*[_ptr(p) for p in ptrs])

    def cp_attention_layers(self, q, k_new, v_new, kv_cache, out, stream=None):
        """q ... out: pointer_array()s of equal length (k_new / v_new may be None)."""
        _check(self.lib.cp_attention_layers(self.handle, len(q), q, k_new, v_new, kv_cache, out, _ptr(stream)))

    def cp_latency_table(self, cap=4096) -> List[cp_latency_row]:
        rows = (cp_latency_row * cap)()
        n = C.c_int32(0)
        _check(self.lib.cp_latency_table(self.handle, rows, cap, C.byref(n)))
        return [rows[i] for i in range(n.value)]

    def cp_set_memory_stats(self, used_mb, free_mb, allocated_mb, reserved_mb):
        _check(self.lib.cp_set_memory_stats(self.handle, used_mb, free_mb, allocated_mb, reserved_mb))

    def cp_get_batch_info(self) -> cp_batch_info:
        info = cp_batch_info()
        _check(self.lib.cp_get_batch_info(self.handle, C.byref(info)))
        return info

    def close(self):
        if self.handle:
            self.lib.cp_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Scheduler:
    """cp_sched_* (host only, no GPU needed)."""

    def __init__(self, alpha=100.0, beta=-1.0, B_max=2048, S_max=1024, mode=CP_MODE_TOKEN_BUDGET,
                 apc=False, Delta=64, T_star=0.0, lambda_u=1.0, lambda_o=2.0, C_max=4, L_min=64,
                 num_blocks=1 << 20, block_size=16, page_mb=0.0625, pred_kind=CP_PRED_LINEAR,
                 pred_weights=None, feat_mu=None, feat_inv_sigma=None, max_batch=None):
        self.lib = load()
        w = np.ascontiguousarray(pred_weights if pred_weights is not None else np.zeros(16), dtype=np.float64)
        mu = np.ascontiguousarray(feat_mu, dtype=np.float64) if feat_mu is not None else None
        inv = np.ascontiguousarray(feat_inv_sigma, dtype=np.float64) if feat_inv_sigma is not None else None
        dp = C.POINTER(C.c_double)
        cfg = cp_sched_config(alpha, beta, B_max, S_max, mode, int(bool(apc)), Delta, C_max, L_min,
                              block_size, num_blocks, T_star, lambda_u, lambda_o, page_mb, pred_kind,
                              len(w), w.ctypes.data_as(dp),
                              mu.ctypes.data_as(dp) if mu is not None else None,
                              inv.ctypes.data_as(dp) if inv is not None else None)
        self.handle = C.c_void_p()
        _check(self.lib.cp_sched_create(C.byref(cfg), C.byref(self.handle)))
        self.cap = max_batch or max(S_max, 1)
        self.descs = (cp_req_desc * self.cap)()
        self.n = 0

    def cp_sched_add_request(self, req_id, arrival_us, prompt_len, output_len):
        _check(self.lib.cp_sched_add_request(self.handle, req_id, arrival_us, prompt_len, output_len))

    def cp_sched_next(self, now_us) -> int:
        """Forms one iteration into self.descs[:n]; returns n."""
        n = C.c_int32(0)
        _check(self.lib.cp_sched_next(self.handle, now_us, self.descs, self.cap, C.byref(n)))
        self.n = n.value
        return self.n

    def batch(self):
        """The formed iteration as [(req_id, q_len, ctx_off, [pages])] (copies)."""
        out = []
        for i in range(self.n):
            d = self.descs[i]
            out.append((d.req_id, d.q_len, d.ctx_off, [d.block_table[k] for k in range(d.n_blocks)]))
        return out

    def cp_sched_commit(self, iter_us):
        _check(self.lib.cp_sched_commit(self.handle, iter_us))

    def cp_sched_next_arrival(self) -> int:
        v = C.c_int64(0)
        _check(self.lib.cp_sched_next_arrival(self.handle, C.byref(v)))
        return v.value

    def cp_sched_has_work(self) -> bool:
        v = C.c_int32(0)
        _check(self.lib.cp_sched_has_work(self.handle, C.byref(v)))
        return bool(v.value)

    def cp_sched_get_stats(self) -> cp_sched_stats:
        st = cp_sched_stats()
        _check(self.lib.cp_sched_get_stats(self.handle, C.byref(st)))
        return st

    def cp_sched_request_times(self, req_id):
        a, b = C.c_int64(0), C.c_int64(0)
        _check(self.lib.cp_sched_request_times(self.handle, req_id, C.byref(a), C.byref(b)))
        return a.value, b.value

    def cp_sched_predict(self, x16) -> float:
        x = np.ascontiguousarray(x16, dtype=np.float64)
        t = C.c_double(0)
        _check(self.lib.cp_sched_predict(self.handle, x.ctypes.data_as(C.POINTER(C.c_double)), C.byref(t)))
        return t.value

    def cp_sched_select_chunk(self, r_i, ctx_i, U_t, n_dec=0, sum_ctx=0, max_ctx=0, pf_tokens=0,
                              n_pf=0, pf_proc=0, pf_proc_max=0) -> int:
        c = C.c_int32(0)
        _check(self.lib.cp_sched_select_chunk(self.handle, r_i, ctx_i, U_t, n_dec, sum_ctx, max_ctx,
                                              pf_tokens, n_pf, pf_proc, pf_proc_max, C.byref(c)))
        return c.value

    def close(self):
        if self.handle:
            self.lib.cp_sched_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
