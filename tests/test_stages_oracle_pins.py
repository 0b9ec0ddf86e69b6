"""Pins of the layer-wise stage oracle (oracle.decode_stages / stage_query, PAPER.md
L126-L128: two in-flight batches, each with its own layer cursor).  CPU only.

P19  alpha = 0 or no dependency: every stage is the (already pinned) single-step attention
P20  the bf16 rounding of the query update, worked by hand (ties to even, both directions)
P21  one-token contexts: O = v exactly, so the next layer's LSE is sigma * <bf16(q + alpha v), k> in closed form
P22  the dependency wiring: a stage sees the output of ITS predecessor, not of the stage listed before it
"""
import numpy as np

import oracle
import workloads as W
from workloads import KIND_KV, ModelCfg

M = ModelCfg(KIND_KV, 8, 2, 128, 128, 128 ** -0.5)


def make(ctxs, seed=3):
    w = W.small_workload([M], [0] * len(ctxs), ctxs, page_tokens=16, seed=seed, keep_contiguous=False)
    rng = np.random.default_rng(seed + 1)
    return w, rng


def rand_q(rng, n):
    return [W.f32_to_bf16(rng.standard_normal((8, 128)).astype(np.float32)) for _ in range(n)]


def test_p19_alpha_zero_and_independent_stages():
    w, rng = make([40, 300, 7, 129])
    stages, deps = [[0, 1], [2, 3], [0, 1], [2, 3]], [-1, -1, 0, 1]
    q_in = [rand_q(rng, 2) for _ in stages]
    got = oracle.decode_stages(w, stages, deps, q_in, alpha=0.0)
    for s, reqs in enumerate(stages):
        for j, ri in enumerate(reqs):
            w.q[ri] = q_in[s][j]
        ref = oracle.decode_workload(w, request_indices=reqs)
        for (o, l), (ro, rl) in zip(got[s], ref):
            assert np.array_equal(o, ro) and np.array_equal(l, rl)
    # without dependencies alpha does not matter
    a = oracle.decode_stages(w, stages, [-1] * 4, q_in, alpha=0.7)
    for s in range(4):
        for (o, l), (ro, rl) in zip(a[s], got[s]):
            assert np.array_equal(o, ro) and np.array_equal(l, rl)


def test_p20_query_update_rounding_by_hand():
    one = np.array([0x3F80], dtype=np.uint16)                       # bf16 1.0, ulp 2^-7
    f = lambda o, a=1.0: int(oracle.stage_query(one, np.array([o], dtype=np.float32), a)[0])
    assert f(0.0) == 0x3F80
    assert f(2.0 ** -8) == 0x3F80                                   # tie, even mantissa below: stays
    assert f(3 * 2.0 ** -8) == 0x3F82                               # tie between odd 0x3F81 and even 0x3F82: up
    assert f(2.0 ** -8 + 2.0 ** -20) == 0x3F81                      # just above the tie
    assert f(2.0 ** -7) == 0x3F81 and f(-2.0 ** -8) == 0x3F7F       # below 1.0 the ulp halves: exact
    assert f(0.5, 2.0) == 0x4000                                    # alpha multiplies O: 1 + 2 * 0.5 = 2
    assert f(1.0, -1.0) == 0x0000                                   # 1 - 1 = +0
    # float32 arithmetic, not float64: 1 + 2^-8 + 2^-30 is a tie in float32 (2^-30 is lost), not above it
    assert f(np.float32(2.0 ** -8) + np.float32(2.0 ** -30)) == 0x3F80


def test_p21_single_token_closed_form():
    w, rng = make([1, 1], seed=9)
    q0, q1 = rand_q(rng, 2), rand_q(rng, 2)
    alpha = 0.5
    got = oracle.decode_stages(w, [[0, 1], [0, 1]], [-1, 0], [q0, q1], alpha)
    for j in range(2):
        r = w.requests[j]
        k, v = oracle.gather(w.arena, 16, w.page_bytes, w.num_pages, KIND_KV, 2, 128, 128, r.page_ids, 1)
        k64, v64 = W.bf16_to_f64(k)[0], W.bf16_to_f64(v)[0]         # [Hkv, 128]
        o0, _ = got[0][j]
        o1, l1 = got[1][j]
        for h in range(8):
            c = h // 4
            assert np.array_equal(o0[h], v64[c]) and np.array_equal(o1[h], v64[c])      # softmax over one token
            q = W.bf16_to_f64(oracle.stage_query(q1[j][h], v64[c].astype(np.float32), alpha))
            np.testing.assert_allclose(l1[h], M.softmax_scale * float(q @ k64[c]), rtol=1e-12, atol=1e-12)


def test_p22_dependency_wiring():
    w, rng = make([200, 64, 200, 64], seed=5)
    stages = [[0, 1], [2, 3], [0, 1]]
    q_in = [rand_q(rng, 2) for _ in stages]
    on0 = oracle.decode_stages(w, stages, [-1, -1, 0], q_in, 1.0)
    on1 = oracle.decode_stages(w, stages, [-1, -1, 1], q_in, 1.0)
    none = oracle.decode_stages(w, stages, [-1, -1, -1], q_in, 1.0)
    assert not np.array_equal(on0[2][0][0], on1[2][0][0]) and not np.array_equal(on0[2][0][0], none[2][0][0])
    # by hand: stage 2 depending on stage 0 is single-step attention with the updated query
    for j, ri in enumerate(stages[2]):
        w.q[ri] = oracle.stage_query(q_in[2][j], on0[0][j][0], 1.0)
    ref = oracle.decode_workload(w, request_indices=stages[2])
    for (o, l), (ro, rl) in zip(on0[2], ref):
        assert np.array_equal(o, ro) and np.array_equal(l, rl)
    # stages 0 and 1 never change
    for s in (0, 1):
        assert np.array_equal(on0[s][0][0], on1[s][0][0]) and np.array_equal(on0[s][1][1], none[s][1][1])
