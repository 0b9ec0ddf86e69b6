"""Pins of oracle.attention_qlen (several query tokens per request, causal; SURVEY §8(f) N4 names the
q_len > 1 variant).  CPU only.

P23  brute force: a dense numpy float64 causal attention with an explicit mask matrix on tiny shapes
P24  q_len = 1 is the single-token oracle; the last token's row never depends on q_len
P25  a query token cannot see later tokens: changing the K/V of a later position leaves its row untouched,
     changing an earlier or its own position does not
"""
import numpy as np

import oracle
import workloads as W
from workloads import KIND_KV, ModelCfg

M = ModelCfg(KIND_KV, 6, 2, 32, 32, 0.2)


def make(ctx, seed):
    w = W.small_workload([M], [0], [ctx], page_tokens=8, seed=seed, keep_contiguous=False)
    r = w.requests[0]
    k, v = oracle.gather(w.arena, 8, w.page_bytes, w.num_pages, KIND_KV, 2, 32, 32, r.page_ids, ctx)
    return w, r, W.bf16_to_f64(k), W.bf16_to_f64(v)


def run(w, r, q):
    return oracle.attention_qlen(w.arena, 8, w.page_bytes, w.num_pages, KIND_KV, 6, 2, 32, 32, 0.2, r.page_ids,
                                 r.context_len, q)


def test_p23_dense_causal_brute_force():
    rng = np.random.default_rng(1)
    for ctx, q_len in ((5, 1), (5, 5), (21, 4), (16, 3), (17, 2)):
        w, r, k, v = make(ctx, seed=10 + ctx)
        q = W.f32_to_bf16(rng.standard_normal((q_len, 6, 32)).astype(np.float32))
        o, lse = run(w, r, q)
        qf = W.bf16_to_f64(q)
        pos = ctx - q_len + np.arange(q_len)                       # position of each query token
        mask = np.arange(ctx)[None, :] <= pos[:, None]             # [q_len, ctx] causal
        for h in range(6):
            c = h // 3
            s = float(np.float32(0.2)) * qf[:, h, :] @ k[:, c, :].T   # [q_len, ctx]; the scale is a float32
            s = np.where(mask, s, -np.inf)
            mx = s.max(axis=1, keepdims=True)
            p = np.exp(s - mx)
            ref = (p @ v[:, c, :]) / p.sum(axis=1, keepdims=True)
            np.testing.assert_allclose(o[:, h, :], ref, rtol=1e-12, atol=1e-14)
            np.testing.assert_allclose(lse[:, h], (mx + np.log(p.sum(axis=1, keepdims=True)))[:, 0], rtol=1e-12)


def test_p24_reduces_to_single_token():
    rng = np.random.default_rng(2)
    w, r, _, _ = make(30, seed=4)
    q = W.f32_to_bf16(rng.standard_normal((4, 6, 32)).astype(np.float32))
    o4, l4 = run(w, r, q)
    o1, l1 = run(w, r, q[3:])
    single = oracle.attention(w.arena, 8, w.page_bytes, w.num_pages, KIND_KV, 6, 2, 32, 32, 0.2, r.page_ids, 30, q[3])
    assert np.array_equal(o4[3], o1[0]) and np.array_equal(l4[3], l1[0])
    assert np.array_equal(o1[0], single[0]) and np.array_equal(l1[0], single[1])


def test_p25_no_token_sees_the_future():
    rng = np.random.default_rng(3)
    ctx, q_len = 19, 4
    w, r, _, _ = make(ctx, seed=6)
    q = W.f32_to_bf16(rng.standard_normal((q_len, 6, 32)).astype(np.float32))
    base_o, base_l = run(w, r, q)
    for pos in (ctx - 1, ctx - 3, ctx - 4, 2):
        w2, r2, _, _ = make(ctx, seed=6)
        k_new = W.f32_to_bf16(rng.standard_normal((2, 32)).astype(np.float32))
        v_new = W.f32_to_bf16(rng.standard_normal((2, 32)).astype(np.float32))
        oracle.append(w2.arena, 8, w2.page_bytes, w2.num_pages, KIND_KV, 2, 32, 32, r2.page_ids, pos, k_new, v_new)
        o, l = run(w2, r2, q)
        for j in range(q_len):
            sees = pos <= ctx - q_len + j
            same = np.array_equal(o[j], base_o[j]) and np.array_equal(l[j], base_l[j])
            assert same != sees, (pos, j)
