"""Seeded synthetic inputs for the paged decode-attention hot path.

This module is the ONLY thing the CPU oracle (`oracle/`) and the CUDA library
(`paper_2606_24506_b200/`) have in common, and it imports neither.  It holds no
attention arithmetic: it draws shapes, context lengths, page assignments and
bf16 values from seeded numpy generators and writes the values into a host
image of the KV arena in the layout `include/crosspool.h` documents
(reading R1 of DESIGN.md: head-granular pages).  Both sides receive the same
host bytes.

The five configurations are the ones `BASELINE.json:configs` lists; they stand
in for the paper's ShareGPT / LongAlign traces, of
which only the context-length mix and the concurrency reach this kernel.  No
dataset item is reproduced anywhere.  The recipe is stated in DESIGN.md §5.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import numpy as np

KIND_KV = 0    # MQA / GQA: separate K rows and V rows
KIND_MLA = 1   # one shared latent row per token; V = its first head_dim_v entries

BF16_NAN = np.uint16(0x7FC0)   # poison written to every unmapped slot (reading A5)

META_SEED_BASE = 2450600
DATA_SEED_BASE = 2451600


@dataclass
class ModelCfg:
    kind: int
    n_q_heads: int
    n_kv_heads: int
    head_dim_qk: int
    head_dim_v: int
    softmax_scale: float          # stored as the float32 value both sides receive

    def __post_init__(self):
        self.softmax_scale = float(np.float32(self.softmax_scale))

    @property
    def group(self) -> int:
        return self.n_q_heads // self.n_kv_heads

    def page_bytes(self, page_tokens: int) -> int:
        if self.kind == KIND_MLA:
            return page_tokens * self.head_dim_qk * 2
        return page_tokens * (self.head_dim_qk + self.head_dim_v) * 2


@dataclass
class Request:
    request_id: int
    model_id: int
    context_len: int
    page_ids: np.ndarray          # int32 [n_logical * n_kv_heads], page-major


@dataclass
class Workload:
    name: str
    page_tokens: int
    page_bytes: int
    num_pages: int
    models: List[ModelCfg]
    requests: List[Request]
    arena: np.ndarray             # uint16 [num_pages * page_bytes / 2]
    q: List[np.ndarray]           # per request uint16 [n_q_heads, head_dim_qk]
    # contiguous copies (only kept on request; used by the gather round-trip pin)
    k_contig: List[Optional[np.ndarray]] = field(default_factory=list)
    v_contig: List[Optional[np.ndarray]] = field(default_factory=list)
    notes: dict = field(default_factory=dict)

    # ---- bookkeeping used by bench / reports (sizes only, no arithmetic of the method)
    def total_tokens(self) -> int:
        return int(sum(r.context_len for r in self.requests))

    def algorithmic_bytes(self) -> int:
        """KV + Q + O + LSE bytes of one decode step."""
        total = 0
        for r in self.requests:
            m = self.models[r.model_id]
            if m.kind == KIND_MLA:
                kv = r.context_len * m.head_dim_qk * 2
            else:
                kv = r.context_len * m.n_kv_heads * (m.head_dim_qk + m.head_dim_v) * 2
            total += kv + m.n_q_heads * m.head_dim_qk * 2 + m.n_q_heads * m.head_dim_v * 4 \
                + m.n_q_heads * 4
        return total

    def flops(self) -> int:
        total = 0
        for r in self.requests:
            m = self.models[r.model_id]
            total += 2 * m.n_q_heads * (m.head_dim_qk + m.head_dim_v) * r.context_len
        return total

    def q_packed(self) -> np.ndarray:
        return np.concatenate([x.reshape(-1) for x in self.q])

    def out_rows(self) -> int:
        return int(sum(self.models[r.model_id].n_q_heads for r in self.requests))


def f32_to_bf16(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit patterns, round-to-nearest-even (no NaN inputs here)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_to_f64(b: np.ndarray) -> np.ndarray:
    """Exact widening of bf16 bit patterns to float64 (for test-side brute force)."""
    u = b.astype(np.uint32) << np.uint32(16)
    return u.view(np.float32).astype(np.float64)


def pages_needed(context_len: int, page_tokens: int) -> int:
    return (context_len + page_tokens - 1) // page_tokens


def scatter_request(arena_pages: np.ndarray, page_tokens: int, model: ModelCfg,
                    page_ids: np.ndarray, k: np.ndarray, v: Optional[np.ndarray]) -> None:
    """Write contiguous K [T,Hkv,dk] (and V [T,Hkv,dv]) bf16 into the arena image.

    arena_pages: uint16 [num_pages, page_bytes/2].  Slots past T in the last page
    keep the poison.  Layout per page (one KV head): K block [P,dk] then V block
    [P,dv]; MLA: one block [P,dk].
    """
    P = page_tokens
    T = k.shape[0]
    hkv = model.n_kv_heads
    n_lp = pages_needed(T, P)
    pm = page_ids.reshape(n_lp, hkv)
    dk = model.head_dim_qk

    def put(block_off: int, rows: np.ndarray, d: int):
        pad = np.full((n_lp * P, hkv, d), BF16_NAN, dtype=np.uint16)
        pad[:T] = rows
        tiles = pad.reshape(n_lp, P, hkv, d).transpose(0, 2, 1, 3).reshape(n_lp * hkv, P * d)
        arena_pages[pm.reshape(-1), block_off:block_off + P * d] = tiles

    put(0, k, dk)
    if model.kind == KIND_KV:
        put(P * dk, v, model.head_dim_v)


def build_workload(name: str, page_tokens: int, models: Sequence[ModelCfg],
                   req_models: Sequence[int], req_ctx: Sequence[int], num_pages: int,
                   page_perm: np.ndarray, data_seed: int, value_scale: float = 1.0,
                   keep_contiguous: bool = False, page_bytes: Optional[int] = None,
                   value_shift: float = 0.0) -> Workload:
    """Assemble a workload: physical pages are consumed from `page_perm` in request
    order (so all models' pages interleave); data drawn per request in the order
    q, K, V (MLA: q, C) from default_rng(data_seed)."""
    models = list(models)
    if page_bytes is None:
        page_bytes = max(m.page_bytes(page_tokens) for m in models)
    assert page_bytes % 2 == 0
    arena = np.full(num_pages * (page_bytes // 2), BF16_NAN, dtype=np.uint16)
    arena_pages = arena.reshape(num_pages, page_bytes // 2)
    rng = np.random.default_rng(data_seed)
    requests: List[Request] = []
    qs, kc, vc = [], [], []
    cursor = 0
    for rid, (mid, T) in enumerate(zip(req_models, req_ctx)):
        m = models[mid]
        T = int(T)
        n_ids = pages_needed(T, page_tokens) * m.n_kv_heads
        ids = np.ascontiguousarray(page_perm[cursor:cursor + n_ids], dtype=np.int32)
        assert ids.size == n_ids, "pool too small for the requested contexts"
        cursor += n_ids
        q = f32_to_bf16(rng.standard_normal((m.n_q_heads, m.head_dim_qk), dtype=np.float32)
                        * np.float32(value_scale))
        k = f32_to_bf16(rng.standard_normal((T, m.n_kv_heads, m.head_dim_qk), dtype=np.float32)
                        * np.float32(value_scale))
        v = None
        if m.kind == KIND_KV:
            v = f32_to_bf16(rng.standard_normal((T, m.n_kv_heads, m.head_dim_v), dtype=np.float32)
                            * np.float32(value_scale) + np.float32(value_shift))
        scatter_request(arena_pages, page_tokens, m, ids, k, v)
        requests.append(Request(rid, int(mid), T, ids))
        qs.append(q)
        if keep_contiguous:
            kc.append(k)
            vc.append(v if v is not None else k[:, :, :m.head_dim_v].copy())
        else:
            kc.append(None)
            vc.append(None)
    return Workload(name, page_tokens, page_bytes, num_pages, models, requests, arena, qs, kc, vc,
                    notes={"data_seed": data_seed, "value_scale": value_scale,
                           "used_pages": cursor})


# --------------------------------------------------------------------------------------
# The five BASELINE.json configurations
# --------------------------------------------------------------------------------------

def _pool_with_slack(total_ids: int) -> int:
    return int(-(-12 * total_ids // 10))      # ceil(1.2 * demand)  (reading A16)


def config1(keep_contiguous: bool = False) -> Workload:
    """Tiny single-model MQA (BASELINE.json configs[0])."""
    k = 1
    rng = np.random.default_rng(META_SEED_BASE + k)
    m = ModelCfg(KIND_KV, 8, 1, 128, 128, 1.0 / np.sqrt(128.0))
    perm = rng.permutation(128)
    return build_workload("cfg1_tiny_mqa", 16, [m], [0, 0], [256, 1000], 128, perm,
                          DATA_SEED_BASE + k, keep_contiguous=keep_contiguous)


def config2_meta():
    k = 2
    rng = np.random.default_rng(META_SEED_BASE + k)
    req_models, req_ctx = [], []
    for mid in range(4):
        n = int(rng.integers(1, 4))
        ctx = rng.integers(4096, 32769, size=n)
        req_models += [mid] * n
        req_ctx += [int(c) for c in ctx]
    return rng, req_models, req_ctx


def config2(keep_contiguous: bool = False) -> Workload:
    """Shared pool of 4 cold GQA models (BASELINE.json configs[1])."""
    rng, req_models, req_ctx = config2_meta()
    models = [ModelCfg(KIND_KV, 32, 4, 128, 128, 1.0 / np.sqrt(128.0)) for _ in range(4)]
    P = 64
    demand = sum(pages_needed(c, P) * 4 for c in req_ctx)
    num_pages = _pool_with_slack(demand)
    perm = rng.permutation(num_pages)
    return build_workload("cfg2_four_gqa", P, models, req_models, req_ctx, num_pages, perm,
                          DATA_SEED_BASE + 2, keep_contiguous=keep_contiguous)


def config3(keep_contiguous: bool = False, ctx=(16384, 32768, 65536, 131072)) -> Workload:
    """MLA latent decode (BASELINE.json configs[2])."""
    k = 3
    rng = np.random.default_rng(META_SEED_BASE + k)
    m = ModelCfg(KIND_MLA, 128, 1, 576, 512, 1.0 / np.sqrt(192.0))
    P = 64
    demand = sum(pages_needed(c, P) for c in ctx)
    num_pages = _pool_with_slack(demand)
    perm = rng.permutation(num_pages)
    return build_workload("cfg3_mla", P, [m], [0] * len(ctx), list(ctx), num_pages, perm,
                          DATA_SEED_BASE + k, value_scale=0.1, keep_contiguous=keep_contiguous)


def config4(keep_contiguous: bool = False, context_len: int = 262144) -> Workload:
    """Bursty long-context MQA, batch 1 (BASELINE.json configs[3])."""
    k = 4
    rng = np.random.default_rng(META_SEED_BASE + k)
    m = ModelCfg(KIND_KV, 32, 1, 128, 128, 1.0 / np.sqrt(128.0))
    perm = rng.permutation(16384)
    return build_workload("cfg4_long_mqa", 64, [m], [0], [context_len], 16384, perm,
                          DATA_SEED_BASE + k, keep_contiguous=keep_contiguous)


def config5_meta(sigma: float = 1.0):
    k = 5
    rng = np.random.default_rng(META_SEED_BASE + k)
    p = np.arange(1, 9, dtype=np.float64) ** -1.1
    p /= p.sum()
    req_models = rng.choice(8, 64, p=p)
    ctx = np.clip(np.rint(np.exp(np.log(2048.0) + sigma * rng.standard_normal(64))), 128, 65536)
    return rng, [int(x) for x in req_models], [int(x) for x in ctx]


def config5(keep_contiguous: bool = False, sigma: float = 1.0) -> Workload:
    """Mixed multi-model batch, one persistent launch (BASELINE.json configs[4])."""
    rng, req_models, req_ctx = config5_meta(sigma)
    models = []
    for i in range(8):
        if i % 2 == 0:
            models.append(ModelCfg(KIND_KV, 64, 8, 128, 128, 1.0 / np.sqrt(128.0)))
        else:
            models.append(ModelCfg(KIND_KV, 16, 1, 128, 128, 1.0 / np.sqrt(128.0)))
    P = 32
    demand = sum(pages_needed(c, P) * models[mid].n_kv_heads
                 for mid, c in zip(req_models, req_ctx))
    num_pages = _pool_with_slack(demand)
    perm = rng.permutation(num_pages)
    w = build_workload("cfg5_mixed", P, models, req_models, req_ctx, num_pages, perm,
                       DATA_SEED_BASE + 5, keep_contiguous=keep_contiguous)
    w.notes["lognormal_sigma"] = sigma
    return w


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def config(k: int, **kw) -> Workload:
    return CONFIGS[k](**kw)


# --------------------------------------------------------------------------------------
# Small free-form workloads for tests
# --------------------------------------------------------------------------------------

def small_workload(models: Sequence[ModelCfg], req_models: Sequence[int], req_ctx: Sequence[int],
                   page_tokens: int, seed: int = 1, extra_pages: int = 7,
                   value_scale: float = 1.0, value_shift: float = 0.0,
                   keep_contiguous: bool = True, name: str = "small") -> Workload:
    models = list(models)
    demand = sum(pages_needed(c, page_tokens) * models[m].n_kv_heads
                 for m, c in zip(req_models, req_ctx))
    num_pages = demand + extra_pages
    rng = np.random.default_rng(seed)
    perm = rng.permutation(num_pages)
    return build_workload(name, page_tokens, models, req_models, req_ctx, num_pages, perm,
                          seed + 1000, value_scale=value_scale, value_shift=value_shift,
                          keep_contiguous=keep_contiguous)
