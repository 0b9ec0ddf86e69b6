"""Pins for the CPU oracle (CPU only).  Each test is chosen so that a plausible mistake
in oracle/cp_oracle.c -- a dropped scale, a wrong sign, a transposed index, a wrong page
or slot, K/V block mix-up, wrong GQA grouping, log base -- fails at least one of them.
Pin names P1..P12 follow SURVEY.md §8(c) / DESIGN.md §3."""
import os
import re
import sys

import numpy as np
import pytest

import oracle
import workloads as W
from workloads import KIND_KV, KIND_MLA, ModelCfg

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------- helpers (test side only)
def bf16(x):
    return W.f32_to_bf16(np.asarray(x, dtype=np.float32))


def dense_reference(q_bits, k_bits, v_bits, sigma, g):
    """Brute force on CONTIGUOUS K/V: softmax(sigma Q K^T) V in numpy float64, built without the
    page table.  q [Hq,dk], k [T,Hkv,dk], v [T,Hkv,dv] as bf16 bit patterns."""
    q = W.bf16_to_f64(q_bits)
    k = W.bf16_to_f64(k_bits)
    v = W.bf16_to_f64(v_bits)
    Hq = q.shape[0]
    out = np.zeros((Hq, v.shape[2]))
    lse = np.zeros(Hq)
    for h in range(Hq):
        c = h // g
        s = sigma * (k[:, c, :] @ q[h])
        m = s.max()
        p = np.exp(s - m)
        out[h] = (p[:, None] * v[:, c, :]).sum(0) / p.sum()
        lse[h] = m + np.log(p.sum())
    return out, lse


def run_oracle(w, i=0, **kw):
    r = w.requests[i]
    m = w.models[r.model_id]
    return oracle.attention(w.arena, w.page_tokens, w.page_bytes, w.num_pages, m.kind, m.n_q_heads,
                            m.n_kv_heads, m.head_dim_qk, m.head_dim_v, m.softmax_scale,
                            r.page_ids, r.context_len, w.q[i], **kw)


def manual_workload(model, page_tokens, q_bits, k_bits, v_bits, seed=3, extra_pages=5):
    """Scatter given contiguous bf16 K/V for ONE request into a fresh poisoned arena."""
    T = k_bits.shape[0]
    n_ids = W.pages_needed(T, page_tokens) * model.n_kv_heads
    num_pages = n_ids + extra_pages
    pb = model.page_bytes(page_tokens)
    arena = np.full(num_pages * pb // 2, W.BF16_NAN, dtype=np.uint16)
    perm = np.random.default_rng(seed).permutation(num_pages)[:n_ids].astype(np.int32)
    W.scatter_request(arena.reshape(num_pages, pb // 2), page_tokens, model, perm, k_bits, v_bits)
    return W.Workload("manual", page_tokens, pb, num_pages, [model],
                      [W.Request(0, 0, T, perm)], arena, [q_bits], [k_bits], [v_bits])


def parse_golden(fn):
    d = {"dots": {}, "out": {}, "out_sigma64": {}}
    for line in open(os.path.join(GOLD, fn)):
        if line.startswith("#") or not line.strip():
            continue
        tok = line.split()
        if tok[0] in ("lse", "lse_sigma64"):
            d[tok[0]] = np.array([float(x) for x in tok[1:]])
        elif tok[0] in ("out", "out_sigma64"):
            d[tok[0]][int(tok[1])] = np.array([float(x) for x in tok[2:]])
        elif tok[0] == "dots":
            d["dots"][int(tok[1])] = tok[2:]
    return d


# ---------------------------------------------------------------- P1 single token
@pytest.mark.parametrize("kind", [KIND_KV, KIND_MLA])
def test_p1_single_token(kind):
    rng = np.random.default_rng(11)
    if kind == KIND_KV:
        m = ModelCfg(KIND_KV, 6, 2, 16, 8, 0.37)
        k = bf16(rng.standard_normal((1, 2, 16)))
        v = bf16(rng.standard_normal((1, 2, 8)))
    else:
        m = ModelCfg(KIND_MLA, 5, 1, 24, 16, 0.37)
        k = bf16(rng.standard_normal((1, 1, 24)))
        v = None
    q = bf16(rng.standard_normal((m.n_q_heads, m.head_dim_qk)))
    w = manual_workload(m, 4, q, k, v)
    out, lse = run_oracle(w)
    vv = W.bf16_to_f64(k[:, :, :m.head_dim_v] if v is None else v)
    for h in range(m.n_q_heads):
        c = h // m.group
        assert np.array_equal(out[h], vv[0, c])          # exactly the value row
        s = m.softmax_scale * float(W.bf16_to_f64(q[h]) @ W.bf16_to_f64(k[0, c]))
        assert abs(lse[h] - s) < 1e-15 * max(1.0, abs(s)) + 1e-15


# ---------------------------------------------------------------- P2 identical keys
def test_p2_identical_keys():
    rng = np.random.default_rng(12)
    T, m = 37, ModelCfg(KIND_KV, 4, 2, 16, 8, 0.25)
    k1 = bf16(rng.standard_normal((1, 2, 16)))
    k = np.repeat(k1, T, axis=0)
    v = bf16(rng.standard_normal((T, 2, 8)))
    q = bf16(rng.standard_normal((4, 16)))
    out, lse = run_oracle(manual_workload(m, 8, q, k, v))
    vv = W.bf16_to_f64(v)
    for h in range(4):
        c = h // 2
        assert np.allclose(out[h], vv[:, c].mean(0), rtol=0, atol=1e-13)
        s = m.softmax_scale * float(W.bf16_to_f64(q[h]) @ W.bf16_to_f64(k1[0, c]))
        assert abs(lse[h] - (s + np.log(T))) < 1e-13


# ---------------------------------------------------------------- P3 two tokens, closed form
def test_p3_two_tokens():
    rng = np.random.default_rng(13)
    m = ModelCfg(KIND_KV, 3, 1, 16, 16, 0.5)
    k = bf16(rng.standard_normal((2, 1, 16)))
    v = bf16(rng.standard_normal((2, 1, 16)))
    q = bf16(rng.standard_normal((3, 16)))
    out, lse = run_oracle(manual_workload(m, 1, q, k, v))   # P = 1: two pages
    kk, vv, qq = W.bf16_to_f64(k), W.bf16_to_f64(v), W.bf16_to_f64(q)
    for h in range(3):
        s0 = m.softmax_scale * float(qq[h] @ kk[0, 0])
        s1 = m.softmax_scale * float(qq[h] @ kk[1, 0])
        wgt = 1.0 / (1.0 + np.exp(s1 - s0))
        assert np.allclose(out[h], wgt * vv[0, 0] + (1 - wgt) * vv[1, 0], rtol=0, atol=1e-14)
        assert abs(lse[h] - np.logaddexp(s0, s1)) < 1e-14


# ---------------------------------------------------------------- P4 V shift / scale
def test_p4_v_affine():
    rng = np.random.default_rng(14)
    T, m = 45, ModelCfg(KIND_KV, 4, 2, 16, 8, 0.3)
    k = bf16(rng.standard_normal((T, 2, 16)))
    # V values on a coarse dyadic grid so that a*V + b is exact in bf16
    v0 = (rng.integers(-8, 9, size=(T, 2, 8)) / 8.0).astype(np.float32)
    a, b = 2.0, (rng.integers(-4, 5, size=(1, 1, 8)) / 4.0).astype(np.float32)
    q = bf16(rng.standard_normal((4, 16)))
    o0, l0 = run_oracle(manual_workload(m, 8, q, k, bf16(v0)))
    o1, l1 = run_oracle(manual_workload(m, 8, q, k, bf16(a * v0 + b)))
    assert np.allclose(o1, a * o0 + b.reshape(1, 8), rtol=0, atol=1e-13)
    assert np.array_equal(l0, l1)


# ---------------------------------------------------------------- P5 page permutation
def test_p5_page_permutation_bit_identical():
    rng = np.random.default_rng(15)
    T, m = 83, ModelCfg(KIND_KV, 8, 4, 16, 16, 0.2)
    k = bf16(rng.standard_normal((T, 4, 16)))
    v = bf16(rng.standard_normal((T, 4, 16)))
    q = bf16(rng.standard_normal((8, 16)))
    ref = run_oracle(manual_workload(m, 8, q, k, v, seed=1))
    for seed in (2, 3, 4):
        got = run_oracle(manual_workload(m, 8, q, k, v, seed=seed, extra_pages=seed * 3))
        assert np.array_equal(ref[0], got[0]) and np.array_equal(ref[1], got[1])


# ---------------------------------------------------------------- P6 split count
@pytest.mark.parametrize("kind", [KIND_KV, KIND_MLA])
def test_p6_split_invariance(kind):
    if kind == KIND_KV:
        m = ModelCfg(KIND_KV, 4, 2, 16, 16, 0.25)
    else:
        m = ModelCfg(KIND_MLA, 4, 1, 24, 16, 0.25)
    w = W.small_workload([m], [0], [75], page_tokens=4, seed=16)
    n_pages = W.pages_needed(75, 4)
    ref = run_oracle(w)
    for ns in (2, 3, 7, n_pages, n_pages + 5):
        got = run_oracle(w, n_splits=ns)
        assert np.allclose(ref[0], got[0], rtol=0, atol=1e-12)
        assert np.allclose(ref[1], got[1], rtol=0, atol=1e-12)


# ---------------------------------------------------------------- P7 batch independence / poison
def test_p7_independent_of_pool_contents():
    m0 = ModelCfg(KIND_KV, 4, 2, 16, 16, 0.25)
    m1 = ModelCfg(KIND_KV, 2, 1, 16, 16, 0.5)
    w = W.small_workload([m0, m1], [0, 1, 0], [29, 50, 7], page_tokens=8, seed=17)
    ref = run_oracle(w, 1)
    mine = set(int(p) for p in w.requests[1].page_ids)
    arena2 = w.arena.copy().reshape(w.num_pages, -1)
    rng = np.random.default_rng(99)
    for p in range(w.num_pages):
        if p not in mine:
            arena2[p] = rng.integers(0, 65536, size=arena2.shape[1]).astype(np.uint16)
    # also rewrite the unused tail of request 1's last page (50 = 6*8 + 2 -> 6 dead slots)
    last = int(w.requests[1].page_ids[-1])
    pg = arena2[last].reshape(2, 8, 16)
    pg[:, 2:, :] = 0x7F81     # signalling-NaN pattern
    w2 = W.Workload("x", w.page_tokens, w.page_bytes, w.num_pages, w.models, w.requests,
                    arena2.reshape(-1), w.q)
    got = run_oracle(w2, 1)
    assert np.array_equal(ref[0], got[0]) and np.array_equal(ref[1], got[1])
    assert np.isfinite(got[0]).all()


# ---------------------------------------------------------------- P8 brute force on tiny shapes
@pytest.mark.parametrize("case", [
    (KIND_KV, 6, 3, 16, 8, 50, 4),      # GQA g=2, dk != dv, partial last page
    (KIND_KV, 5, 1, 8, 16, 33, 16),     # MQA, dv > dk
    (KIND_KV, 4, 4, 16, 16, 17, 1),     # MHA, P = 1
    (KIND_MLA, 7, 1, 16, 12, 41, 8),    # MLA, V = first 12 of 16
    (KIND_MLA, 3, 1, 6, 4, 9, 2),
])
def test_p8_brute_force_dense(case):
    kind, hq, hkv, dk, dv, T, P = case
    m = ModelCfg(kind, hq, hkv, dk, dv, 1.0 / np.sqrt(dk))
    w = W.small_workload([m], [0], [T], page_tokens=P, seed=18 + T)
    out, lse = run_oracle(w)
    ro, rl = dense_reference(w.q[0], w.k_contig[0], w.v_contig[0], m.softmax_scale, m.group)
    assert np.allclose(out, ro, rtol=0, atol=1e-13)
    assert np.allclose(lse, rl, rtol=0, atol=1e-13)


def test_p8_multi_request_mixed_models():
    ms = [ModelCfg(KIND_KV, 8, 2, 16, 16, 0.25), ModelCfg(KIND_KV, 4, 1, 16, 16, 0.25)]
    w = W.small_workload(ms, [0, 1, 1, 0], [13, 64, 5, 31], page_tokens=8, seed=21)
    res = oracle.decode_workload(w)
    for i, (out, lse) in enumerate(res):
        m = ms[w.requests[i].model_id]
        ro, rl = dense_reference(w.q[i], w.k_contig[i], w.v_contig[i], m.softmax_scale, m.group)
        assert np.allclose(out, ro, rtol=0, atol=1e-13) and np.allclose(lse, rl, rtol=0, atol=1e-13)


# ---------------------------------------------------------------- P9 GQA = replicated MQA
def test_p9_gqa_equals_mqa_per_kv_head():
    rng = np.random.default_rng(22)
    T, hq, hkv, d = 39, 8, 4, 16
    g = hq // hkv
    k = bf16(rng.standard_normal((T, hkv, d)))
    v = bf16(rng.standard_normal((T, hkv, d)))
    q = bf16(rng.standard_normal((hq, d)))
    out, lse = run_oracle(manual_workload(ModelCfg(KIND_KV, hq, hkv, d, d, 0.25), 8, q, k, v))
    for c in range(hkv):
        mq = ModelCfg(KIND_KV, g, 1, d, d, 0.25)
        o1, l1 = run_oracle(manual_workload(mq, 8, q[c * g:(c + 1) * g], k[:, c:c + 1], v[:, c:c + 1]))
        assert np.array_equal(out[c * g:(c + 1) * g], o1) and np.array_equal(lse[c * g:(c + 1) * g], l1)


# ---------------------------------------------------------------- P10 MLA = KV kind with V aliasing K
def test_p10_mla_equals_kv_with_aliased_v():
    rng = np.random.default_rng(23)
    T, hq, w_, dv = 52, 6, 24, 16
    c = bf16(rng.standard_normal((T, 1, w_)) * 0.3)
    q = bf16(rng.standard_normal((hq, w_)))
    o_mla = run_oracle(manual_workload(ModelCfg(KIND_MLA, hq, 1, w_, dv, 0.2), 8, q, c, None))
    o_kv = run_oracle(manual_workload(ModelCfg(KIND_KV, hq, 1, w_, dv, 0.2), 8, q, c,
                                      np.ascontiguousarray(c[:, :, :dv])))
    assert np.array_equal(o_mla[0], o_kv[0]) and np.array_equal(o_mla[1], o_kv[1])


# ---------------------------------------------------------------- P11 golden vectors
def _g1_inputs():
    Q = np.array([[(((7 * h + 3 * i) % 5) - 2) / 2 for i in range(8)] for h in range(2)], np.float32)
    K = np.array([[(((5 * t + 11 * i) % 7) - 3) / 4 for i in range(8)] for t in range(5)], np.float32)
    V = np.array([[(((4 * t + 5 * i) % 9) - 4) / 8 for i in range(8)] for t in range(5)], np.float32)
    return Q, K, V


def _g2_inputs():
    Q = np.array([[(((5 * h + 2 * i) % 7) - 3) / 4 for i in range(6)] for h in range(3)], np.float32)
    C = np.array([[(((3 * t + 5 * i) % 11) - 5) / 8 for i in range(6)] for t in range(4)], np.float32)
    return Q, C


def test_p11_golden_g1():
    Q, K, V = _g1_inputs()
    m = ModelCfg(KIND_KV, 2, 1, 8, 8, 1.0 / np.sqrt(8.0))
    w = manual_workload(m, 2, bf16(Q), bf16(K).reshape(5, 1, 8), bf16(V).reshape(5, 1, 8))
    assert np.array_equal(W.bf16_to_f64(w.q[0]), Q.astype(np.float64))   # inputs exact in bf16
    out, lse = run_oracle(w)
    g = parse_golden("g1_kv.txt")
    assert np.allclose(lse, g["lse"], rtol=0, atol=1e-11)
    for h in range(2):
        assert np.allclose(out[h], g["out"][h], rtol=0, atol=1e-11)
        # SURVEY's printed digits use the unrounded sigma; fp32 rounding of sigma moves
        # the result by <= |d sigma| * max|q.k| ~ 6e-9 * 2.75
        assert np.allclose(out[h], g["out_sigma64"][h], rtol=0, atol=2e-8)
    assert np.allclose(lse, g["lse_sigma64"], rtol=0, atol=2e-8)


def test_p11_golden_g2():
    Q, C = _g2_inputs()
    m = ModelCfg(KIND_MLA, 3, 1, 6, 4, 1.0 / np.sqrt(3.0))
    out, lse = run_oracle(manual_workload(m, 2, bf16(Q), bf16(C).reshape(4, 1, 6), None))
    g = parse_golden("g2_mla.txt")
    assert np.allclose(lse, g["lse"], rtol=0, atol=1e-11)
    for h in range(3):
        assert np.allclose(out[h], g["out"][h], rtol=0, atol=1e-11)
        assert np.allclose(out[h], g["out_sigma64"][h], rtol=0, atol=2e-8)


def test_golden_files_rederive():
    """The committed fixtures are exactly what tests/golden/make_golden.py derives, and
    its unrounded-sigma lines carry the digits printed in SURVEY.md §8(c)."""
    sys.path.insert(0, GOLD)
    import make_golden
    texts = make_golden.main(write=False)
    for fn, t in texts.items():
        assert open(os.path.join(GOLD, fn)).read() == t
    g = parse_golden("g1_kv.txt")
    assert g["dots"][0] == ["5/4", "-7/4", "-3/8", "11/4", "-9/8"]
    assert g["dots"][1] == ["-11/8", "5/8", "7/8", "-3/2", "-3/8"]
    assert list(g["lse_sigma64"]) == [1.838319507914, 1.545236062785]
    assert list(g["out_sigma64"][0][:3]) == [-0.066577421388, 0.185037856673, -0.098324929982]
    g2 = parse_golden("g2_mla.txt")
    assert g2["dots"][2] == ["-1/2", "3/8", "-1/8", "-5/8"]
    assert list(g2["lse_sigma64"]) == [1.519434505815, 1.476856889790, 1.286045256556]
    assert list(g2["out_sigma64"][1]) == [0.023513673560, -0.201379766413, 0.212500842024,
                                          0.056536475348]


# ---------------------------------------------------------------- P12 gather round trip
@pytest.mark.parametrize("kind", [KIND_KV, KIND_MLA])
def test_p12_gather_round_trip(kind):
    if kind == KIND_KV:
        ms = [ModelCfg(KIND_KV, 8, 4, 16, 8, 0.25), ModelCfg(KIND_KV, 2, 1, 16, 8, 0.25)]
        w = W.small_workload(ms, [0, 1, 0], [37, 64, 1], page_tokens=8, seed=31)
    else:
        ms = [ModelCfg(KIND_MLA, 4, 1, 24, 16, 0.25)]
        w = W.small_workload(ms, [0, 0], [19, 33], page_tokens=4, seed=32)
    # include awkward bit patterns in the data: -0.0, NaN payloads, denormals
    r0 = w.requests[0]
    m0 = ms[r0.model_id]
    for i, r in enumerate(w.requests):
        m = ms[r.model_id]
        k, v = oracle.gather(w.arena, w.page_tokens, w.page_bytes, w.num_pages, m.kind,
                             m.n_kv_heads, m.head_dim_qk, m.head_dim_v, r.page_ids, r.context_len)
        assert k.tobytes() == w.k_contig[i].tobytes()
        assert v.tobytes() == w.v_contig[i].tobytes()
        assert not (k == W.BF16_NAN).any()     # never returns a poisoned slot


def test_p12_gather_special_bit_patterns():
    m = ModelCfg(KIND_KV, 2, 2, 8, 8, 1.0)
    rng = np.random.default_rng(5)
    k = rng.integers(0, 65536, size=(21, 2, 8)).astype(np.uint16)   # any pattern incl. NaN/-0
    v = rng.integers(0, 65536, size=(21, 2, 8)).astype(np.uint16)
    k[0, 0, 0], k[0, 0, 1], v[3, 1, 2] = 0x8000, 0x7FA5, 0x0001
    w = manual_workload(m, 4, bf16(np.zeros((2, 8))), k, v)
    r = w.requests[0]
    gk, gv = oracle.gather(w.arena, 4, w.page_bytes, w.num_pages, KIND_KV, 2, 8, 8, r.page_ids, 21)
    assert gk.tobytes() == k.tobytes() and gv.tobytes() == v.tobytes()


# ---------------------------------------------------------------- P13 append
@pytest.mark.parametrize("kind", [KIND_KV, KIND_MLA])
def test_p13_append_token_by_token(kind):
    """Building a request with the oracle's append, one token at a time into an all-poison arena,
    gives exactly the arena a direct scatter gives: the expected image is written here with the
    address formula of DESIGN.md §4 (numpy indexing, not the oracle), compared byte for byte, so
    every other byte must still be poison."""
    P = 4
    if kind == KIND_KV:
        Hkv, dk, dv = 3, 16, 8
        page_u16 = P * (dk + dv)
    else:
        Hkv, dk, dv = 1, 24, 16
        page_u16 = P * dk
    T, num_pages = 11, 20
    rng = np.random.default_rng(77)
    n_lp = -(-T // P)
    page_ids = rng.permutation(num_pages)[:n_lp * Hkv].astype(np.int32)
    k = rng.integers(0, 65536, size=(T, Hkv, dk)).astype(np.uint16)
    v = rng.integers(0, 65536, size=(T, Hkv, dv)).astype(np.uint16)
    arena = np.full(num_pages * page_u16, W.BF16_NAN, dtype=np.uint16)
    expect = arena.copy().reshape(num_pages, page_u16)
    for t in range(T):
        oracle.append(arena, P, page_u16 * 2, num_pages, kind, Hkv, dk, dv, page_ids, t, k[t],
                      None if kind == KIND_MLA else v[t])
        for c in range(Hkv):
            pg = expect[page_ids[(t // P) * Hkv + c]]
            pg[(t % P) * dk:(t % P) * dk + dk] = k[t, c]
            if kind == KIND_KV:
                pg[P * dk + (t % P) * dv:P * dk + (t % P) * dv + dv] = v[t, c]
        assert arena.tobytes() == expect.tobytes()
    gk, gv = oracle.gather(arena, P, page_u16 * 2, num_pages, kind, Hkv, dk, dv, page_ids, T)
    assert gk.tobytes() == k.tobytes()
    if kind == KIND_KV:
        assert gv.tobytes() == v.tobytes()
    else:
        assert gv.tobytes() == np.ascontiguousarray(k[:, :, :dv]).tobytes()
    with pytest.raises(ValueError):          # page list does not cover the position
        oracle.append(arena, P, page_u16 * 2, num_pages, kind, Hkv, dk, dv, page_ids, n_lp * P, k[0],
                      None if kind == KIND_MLA else v[0])


# ---------------------------------------------------------------- argument checks
def test_oracle_rejects_bad_arguments():
    m = ModelCfg(KIND_KV, 4, 2, 16, 16, 0.25)
    w = W.small_workload([m], [0], [20], page_tokens=8, seed=40)
    r = w.requests[0]
    with pytest.raises(ValueError):
        oracle.attention(w.arena, 8, w.page_bytes, w.num_pages, KIND_KV, 4, 2, 16, 16, 0.25,
                         r.page_ids[:2], 20, w.q[0])                 # too few pages
    bad = r.page_ids.copy()
    bad[0] = w.num_pages
    with pytest.raises(ValueError):
        oracle.attention(w.arena, 8, w.page_bytes, w.num_pages, KIND_KV, 4, 2, 16, 16, 0.25,
                         bad, 20, w.q[0])                             # page id out of range
    with pytest.raises(ValueError):
        oracle.attention(w.arena, 8, w.page_bytes, w.num_pages, KIND_KV, 4, 3, 16, 16, 0.25,
                         r.page_ids, 20, w.q[0])                      # Hq % Hkv != 0


# ---------------------------------------------------------------- generator anchors
def test_generator_anchors():
    """The seeded recipe of DESIGN.md §5 reproduces the check draws recorded in SURVEY.md §8(d)."""
    assert list(np.random.default_rng(2450601).permutation(128)[:8]) == [124, 48, 52, 36, 95, 7, 122, 94]
    _, rm, rc = W.config2_meta()
    assert rm == [0, 0, 1, 2, 2, 3, 3, 3]
    assert rc == [27786, 12973, 14815, 31836, 24658, 30242, 4959, 20636]
    _, rm5, rc5 = W.config5_meta()
    assert list(np.bincount(rm5, minlength=8)) == [26, 12, 11, 4, 6, 0, 2, 3]
    assert (min(rc5), max(rc5), sum(rc5)) == (245, 45279, 226374)
    w1 = W.config1()
    assert w1.algorithmic_bytes() == 643072 + 4096 + 8192 + 64
    assert int(w1.requests[1].page_ids[-1]) == 0
    # poison everywhere outside mapped slots: tail of request 1's last page
    pg = w1.arena.reshape(128, -1)[0].reshape(2, 16, 128)
    assert (pg[:, 8:, :] == W.BF16_NAN).all() and not (pg[:, :8, :] == W.BF16_NAN).any()
