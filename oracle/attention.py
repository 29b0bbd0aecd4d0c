"""ctypes front end of the fp64 C oracle (TEST INFRASTRUCTURE, not product code).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
leg may import this.  It imports nothing from paper_2606_09061_b200.

Definition followed: SURVEY.md 8(c1) -- textbook causal softmax attention over a
paged KV cache (PAPER.md:41 paged attention; PAPER.md:61, :87 mixed batch of
decodes + prefill chunks).  All arrays are numpy; bf16 tensors travel as uint16
bit patterns.  Cache layout: kv_cache[block][2][Hkv][B][D] (one layer).
"""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        lib.oracle_num_threads.restype = C.c_int
        lib.oracle_kv_append.restype = C.c_int
        lib.oracle_attention_rows.restype = C.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _p(a, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def _flatten_tables(block_tables):
    bt_off = np.zeros(len(block_tables) + 1, dtype=np.int32)
    for j, bt in enumerate(block_tables):
        bt_off[j + 1] = bt_off[j] + len(bt)
    flat = (np.concatenate([np.asarray(b, dtype=np.int32) for b in block_tables])
            if len(block_tables) else np.zeros(0, dtype=np.int32))
    return bt_off, np.ascontiguousarray(flat, dtype=np.int32)


def kv_append(k_new, v_new, kv_cache, q_len, ctx_off, block_tables):
    """Write this iteration's K/V rows into their pages, in place (H2).

    k_new, v_new: uint16 [T, Hkv, D]; kv_cache: uint16 [num_blocks, 2, Hkv, B, D].
    """
    lib = _load()
    assert kv_cache.dtype == np.uint16 and kv_cache.flags.c_contiguous
    num_blocks, two, Hkv, B, D = kv_cache.shape
    assert two == 2
    k_new = np.ascontiguousarray(k_new, dtype=np.uint16)
    v_new = np.ascontiguousarray(v_new, dtype=np.uint16)
    q_len = np.ascontiguousarray(q_len, dtype=np.int32)
    ctx_off = np.ascontiguousarray(ctx_off, dtype=np.int32)
    bt_off, flat = _flatten_tables(block_tables)
    rc = lib.oracle_kv_append(
        _p(k_new, C.c_uint16), _p(v_new, C.c_uint16), _p(kv_cache, C.c_uint16),
        _p(q_len, C.c_int32), _p(ctx_off, C.c_int32), _p(bt_off, C.c_int32),
        _p(flat, C.c_int32), C.c_int(len(q_len)), C.c_int(Hkv), C.c_int(D),
        C.c_int(B), C.c_int64(num_blocks))
    if rc != 0:
        raise ValueError("oracle_kv_append: bad block table")


def attention(q, kv_cache, q_len, ctx_off, block_tables, sm_scale,
              rows=None):
    """fp64 attention output.

    q: uint16 [T, Hq, D]; kv_cache as above, ALREADY holding this iteration's K/V.
    rows: None -> all rows, returns float64 [T, Hq, D];
          else (tok[int64 n], head[int32 n]) -> returns float64 [n, D].
    sm_scale is used as float32 widened to fp64 (the constant the GPU receives).
    """
    lib = _load()
    assert q.dtype == np.uint16 and kv_cache.dtype == np.uint16
    q = np.ascontiguousarray(q)
    assert kv_cache.flags.c_contiguous
    T, Hq, D = q.shape
    num_blocks, two, Hkv, B, Dc = kv_cache.shape
    assert two == 2 and Dc == D
    q_len = np.ascontiguousarray(q_len, dtype=np.int32)
    ctx_off = np.ascontiguousarray(ctx_off, dtype=np.int32)
    assert int(q_len.sum()) == T
    bt_off, flat = _flatten_tables(block_tables)
    scale = float(np.float32(sm_scale))
    if rows is None:
        out = np.empty((T, Hq, D), dtype=np.float64)
        tok_p, head_p, n_rows = None, None, T * Hq
    else:
        tok = np.ascontiguousarray(rows[0], dtype=np.int64)
        head = np.ascontiguousarray(rows[1], dtype=np.int32)
        assert tok.shape == head.shape
        out = np.empty((len(tok), D), dtype=np.float64)
        tok_p, head_p, n_rows = _p(tok, C.c_int64), _p(head, C.c_int32), len(tok)
    rc = lib.oracle_attention_rows(
        _p(q, C.c_uint16), _p(kv_cache, C.c_uint16), _p(q_len, C.c_int32),
        _p(ctx_off, C.c_int32), _p(bt_off, C.c_int32), _p(flat, C.c_int32),
        C.c_int(len(q_len)), C.c_int(Hq), C.c_int(Hkv), C.c_int(D), C.c_int(B),
        C.c_int64(num_blocks), C.c_double(scale), tok_p, head_p,
        C.c_int64(n_rows), _p(out, C.c_double))
    if rc != 0:
        raise ValueError("oracle_attention_rows: bad arguments / block table")
    return out


def combine_partials(m, l, o):
    """LSE merge of per-range softmax partials.

    m [S], l [S], o [S, D]: for split s over key range R_s, m_s = max score,
    l_s = sum exp(score - m_s), o_s = sum exp(score - m_s) v  (unnormalised).
    Empty ranges carry m = -inf, l = 0, o = 0.  Returns the normalised output:
      M = max_s m_s ; w_s = exp(m_s - M) ; out = sum_s w_s o_s / sum_s w_s l_s.
    """
    m = np.asarray(m, dtype=np.float64)
    l = np.asarray(l, dtype=np.float64)
    o = np.asarray(o, dtype=np.float64)
    M = np.max(m)
    w = np.where(np.isneginf(m), 0.0, np.exp(m - M))
    return (w[:, None] * o).sum(axis=0) / (w * l).sum()
