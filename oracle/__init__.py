"""ctypes front end of the CPU float64 oracle (`oracle/cp_oracle.c`).

TEST INFRASTRUCTURE ONLY: importable from tests/, `__graft_entry__.smoke()` and
`bench.py`'s cpu_baseline / `--impl reference` legs.  Nothing under
`paper_2606_24506_b200/` may import it, and it imports nothing from there.
The attention, gather, append and planner arithmetic is in the C file; this file marshals arguments and holds
the three pieces written in numpy / Python loops (each pinned like the C parts): `stage_query` / `_bf16_round`
(bf16 rounding of a dependent stage's query, pin P20), the stage loop of `decode_stages` (P19, P21, P22) and the
per-query-token loop of `attention_qlen` (P23-P25).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cp_oracle.c")
_LIB = os.path.join(_HERE, "libcp_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               "-Wall", "-Wextra", _SRC, "-o", tmp, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        u16p = ctypes.POINTER(ctypes.c_uint16)
        i32p = ctypes.POINTER(ctypes.c_int32)
        f64p = ctypes.POINTER(ctypes.c_double)
        L.cpo_num_threads.restype = ctypes.c_int
        L.cpo_gather.restype = ctypes.c_int
        L.cpo_gather.argtypes = [u16p, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32,
                                 ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                 i32p, ctypes.c_int, ctypes.c_int, u16p, u16p]
        L.cpo_append.restype = ctypes.c_int
        L.cpo_append.argtypes = [u16p, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32,
                                 ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                 i32p, ctypes.c_int, ctypes.c_int, u16p, u16p]
        L.cpo_attention.restype = ctypes.c_int
        L.cpo_attention.argtypes = [u16p, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32,
                                    ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                    ctypes.c_int, ctypes.c_float,
                                    i32p, ctypes.c_int, ctypes.c_int,
                                    u16p, i32p, ctypes.c_int, ctypes.c_int, f64p, f64p]
        i64p = ctypes.POINTER(ctypes.c_int64)
        L.cpo_active_tokens.restype = ctypes.c_double
        L.cpo_active_tokens.argtypes = [ctypes.c_double] * 4
        L.cpo_pool_demand.restype = ctypes.c_int
        L.cpo_pool_demand.argtypes = [ctypes.c_int, i64p, f64p, f64p, f64p, f64p, f64p, ctypes.c_int64, f64p, f64p]
        L.cpo_quantile.restype = ctypes.c_int
        L.cpo_quantile.argtypes = [f64p, ctypes.c_int64, ctypes.c_double, f64p, f64p]
        L.cpo_page_budget.restype = ctypes.c_int64
        L.cpo_page_budget.argtypes = [ctypes.c_double, ctypes.c_double]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().cpo_num_threads())


def _p(a: np.ndarray, ty):
    return a.ctypes.data_as(ctypes.POINTER(ty))


def gather(arena: np.ndarray, page_tokens: int, page_bytes: int, num_pages: int, kind: int,
           n_kv_heads: int, d_k: int, d_v: int, page_ids: np.ndarray, context_len: int):
    """-> (K uint16 [T,Hkv,d_k], V uint16 [T,Hkv,d_v]) bit patterns."""
    arena = np.ascontiguousarray(arena, dtype=np.uint16)
    page_ids = np.ascontiguousarray(page_ids, dtype=np.int32)
    k = np.empty((context_len, n_kv_heads, d_k), dtype=np.uint16)
    v = np.empty((context_len, n_kv_heads, d_v), dtype=np.uint16)
    rc = lib().cpo_gather(_p(arena, ctypes.c_uint16), page_tokens, page_bytes, num_pages, kind,
                          n_kv_heads, d_k, d_v, _p(page_ids, ctypes.c_int32), page_ids.size,
                          context_len, _p(k, ctypes.c_uint16), _p(v, ctypes.c_uint16))
    if rc != 0:
        raise ValueError("cpo_gather failed: %d" % rc)
    return k, v


def append(arena: np.ndarray, page_tokens: int, page_bytes: int, num_pages: int, kind: int,
           n_kv_heads: int, d_k: int, d_v: int, page_ids: np.ndarray, pos: int,
           k_new: np.ndarray, v_new: Optional[np.ndarray]):
    """Write one new token's rows at position `pos` IN PLACE into `arena` (uint16, C-contiguous)."""
    assert arena.dtype == np.uint16 and arena.flags["C_CONTIGUOUS"]
    page_ids = np.ascontiguousarray(page_ids, dtype=np.int32)
    k_new = np.ascontiguousarray(k_new, dtype=np.uint16)
    vp = None
    if v_new is not None:
        v_new = np.ascontiguousarray(v_new, dtype=np.uint16)
        vp = _p(v_new, ctypes.c_uint16)
    rc = lib().cpo_append(_p(arena, ctypes.c_uint16), page_tokens, page_bytes, num_pages, kind,
                          n_kv_heads, d_k, d_v, _p(page_ids, ctypes.c_int32), page_ids.size, pos,
                          _p(k_new, ctypes.c_uint16), vp)
    if rc != 0:
        raise ValueError("cpo_append failed: %d" % rc)


def attention(arena: np.ndarray, page_tokens: int, page_bytes: int, num_pages: int, kind: int,
              n_q_heads: int, n_kv_heads: int, d_k: int, d_v: int, softmax_scale: float,
              page_ids: np.ndarray, context_len: int, q: np.ndarray,
              heads: Optional[Sequence[int]] = None, n_splits: int = 1):
    """-> (O float64 [n_sel, d_v], LSE float64 [n_sel]) for one request."""
    arena = np.ascontiguousarray(arena, dtype=np.uint16)
    page_ids = np.ascontiguousarray(page_ids, dtype=np.int32)
    q = np.ascontiguousarray(q, dtype=np.uint16)
    assert q.size == n_q_heads * d_k
    if heads is None:
        n_sel, hp = n_q_heads, None
    else:
        h = np.ascontiguousarray(heads, dtype=np.int32)
        n_sel, hp = h.size, _p(h, ctypes.c_int32)
    out = np.empty((n_sel, d_v), dtype=np.float64)
    lse = np.empty((n_sel,), dtype=np.float64)
    rc = lib().cpo_attention(_p(arena, ctypes.c_uint16), page_tokens, page_bytes, num_pages, kind,
                             n_q_heads, n_kv_heads, d_k, d_v, ctypes.c_float(softmax_scale),
                             _p(page_ids, ctypes.c_int32), page_ids.size, context_len,
                             _p(q, ctypes.c_uint16), hp, n_sel, n_splits,
                             _p(out, ctypes.c_double), _p(lse, ctypes.c_double))
    if rc != 0:
        raise ValueError("cpo_attention failed: %d" % rc)
    return out, lse


def decode_workload(w, heads_per_request: Optional[Sequence[Optional[Sequence[int]]]] = None,
                    request_indices: Optional[Sequence[int]] = None, n_splits: int = 1):
    """Run the oracle over (a subset of) a `workloads.Workload`, request by request.

    Returns a list of (O, LSE) per selected request.  `w` is duck-typed so that this
    module need not import the generator.
    """
    res = []
    idx = range(len(w.requests)) if request_indices is None else request_indices
    for n, i in enumerate(idx):
        r = w.requests[i]
        m = w.models[r.model_id]
        heads = None if heads_per_request is None else heads_per_request[n]
        res.append(attention(w.arena, w.page_tokens, w.page_bytes, w.num_pages, m.kind,
                             m.n_q_heads, m.n_kv_heads, m.head_dim_qk, m.head_dim_v,
                             m.softmax_scale, r.page_ids, r.context_len, w.q[i],
                             heads=heads, n_splits=n_splits))
    return res


# ---------------------------------------------------------------- several query tokens per request (q_len > 1)
def attention_qlen(arena, page_tokens: int, page_bytes: int, num_pages: int, kind: int, n_q_heads: int,
                   n_kv_heads: int, d_k: int, d_v: int, softmax_scale: float, page_ids, context_len: int,
                   q: np.ndarray):
    """Causal attention of the LAST q_len tokens of a request (reading Q1): q is bf16 bits
    [q_len, Hq, d_k]; query token j sits at position context_len - q_len + j (its own K/V is already in
    the pool and counted by context_len) and attends to positions 0 .. context_len - q_len + j.  That
    is, by definition, the single-token attention over the prefix that ends with token j.
    -> (O float64 [q_len, Hq, d_v], LSE float64 [q_len, Hq])."""
    q = np.ascontiguousarray(q, dtype=np.uint16)
    q_len = q.shape[0]
    assert 1 <= q_len <= context_len
    out = np.empty((q_len, n_q_heads, d_v), dtype=np.float64)
    lse = np.empty((q_len, n_q_heads), dtype=np.float64)
    for j in range(q_len):
        out[j], lse[j] = attention(arena, page_tokens, page_bytes, num_pages, kind, n_q_heads, n_kv_heads, d_k,
                                   d_v, softmax_scale, page_ids, context_len - q_len + 1 + j, q[j])
    return out, lse


# ---------------------------------------------------------------- layer-wise stages
def _bf16_round(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit patterns, round to nearest, ties to even (finite inputs)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    return ((u + 0x7FFF + ((u >> 16) & 1)) >> 16).astype(np.uint16)


def _bf16_widen(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def stage_query(q_in: np.ndarray, o_prev: np.ndarray, alpha: float) -> np.ndarray:
    """Query of a dependent stage (reading M1): the attention output of the layer
    before comes back through the (mocked) FFN as a residual, q = bf16(fp32(q_in) + alpha * O_prev),
    one float32 product and one float32 sum, then round-to-nearest-even."""
    prod = np.float32(alpha) * np.ascontiguousarray(o_prev, dtype=np.float32)
    return _bf16_round(_bf16_widen(q_in) + prod)


def decode_stages(w, stages: Sequence[Sequence[int]], deps: Sequence[int], q_in, alpha: float):
    """Attention-only mock of the layer-wise pipeline: stage s is one attention step (one layer of one
    in-flight batch) over the requests `stages[s]` (indices into w.requests) with queries q_in[s][j]
    (bf16 bits [Hq, d_k]); if deps[s] >= 0 the query first takes the output of stage deps[s] (same
    batch shape) through `stage_query`.  Stages are evaluated one after the other in list order.
    Returns per stage a list of (O, LSE)."""
    outs = []
    for s, reqs in enumerate(stages):
        res = []
        for j, ri in enumerate(reqs):
            r = w.requests[ri]
            m = w.models[r.model_id]
            q = np.ascontiguousarray(q_in[s][j], dtype=np.uint16)
            if deps[s] >= 0:
                assert deps[s] < s and m.head_dim_qk == m.head_dim_v
                q = stage_query(q, outs[deps[s]][j][0], alpha)
            res.append(attention(w.arena, w.page_tokens, w.page_bytes, w.num_pages, m.kind, m.n_q_heads,
                                 m.n_kv_heads, m.head_dim_qk, m.head_dim_v, m.softmax_scale, r.page_ids,
                                 r.context_len, q))
        outs.append(res)
    return outs


# ---------------------------------------------------------------- KV-cache planner (Eq. (1)-(2))
def active_tokens(u: float, o_p: float, o_d: float, t_res: float) -> float:
    """Q_i(u) of Eq. (1)."""
    return float(lib().cpo_active_tokens(float(u), float(o_p), float(o_d), float(t_res)))


def pool_demand(offsets, kappa, arrival, o_p, o_d, t_res, t_obs) -> np.ndarray:
    """K_pool(t) of Eq. (1)-(2) at every observation time (bytes, float64).  Model M owns trace
    entries offsets[M] .. offsets[M+1]-1."""
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in (kappa, arrival, o_p, o_d, t_res, t_obs)]
    kappa, arrival, o_p, o_d, t_res, t_obs = arrs
    assert offsets.size == kappa.size + 1 and offsets[-1] == arrival.size == o_p.size == o_d.size == t_res.size
    out = np.empty(t_obs.size, dtype=np.float64)
    rc = lib().cpo_pool_demand(kappa.size, _p(offsets, ctypes.c_int64), _p(kappa, ctypes.c_double),
                               _p(arrival, ctypes.c_double), _p(o_p, ctypes.c_double), _p(o_d, ctypes.c_double),
                               _p(t_res, ctypes.c_double), t_obs.size, _p(t_obs, ctypes.c_double),
                               _p(out, ctypes.c_double))
    if rc != 0:
        raise ValueError("cpo_pool_demand failed: %d" % rc)
    return out


def quantile(x, q: float) -> float:
    """Empirical quantile x_(ceil(q n)) (no interpolation)."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    scratch = np.empty_like(x)
    out = ctypes.c_double()
    rc = lib().cpo_quantile(_p(x, ctypes.c_double), x.size, float(q), _p(scratch, ctypes.c_double), ctypes.byref(out))
    if rc != 0:
        raise ValueError("cpo_quantile failed: %d" % rc)
    return float(out.value)


def page_budget(k_bytes: float, page_bytes: float) -> int:
    return int(lib().cpo_page_budget(float(k_bytes), float(page_bytes)))
