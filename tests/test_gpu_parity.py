"""GPU parity tests (run with -m gpu on the B200 box): the CUDA path, called through the
C ABI, against the CPU float64 oracle on the same seeded inputs.

Bars (BASELINE.json north_star / DESIGN.md §3): translation + gather bit-exact; attention
max-abs <= 1e-2 and mean-abs <= 1e-3 over all outputs of a config, LSE max-abs <= 1e-3, and
the self-imposed per-request relative bound ||dO||_F / ||O*||_F <= 1e-2 (the absolute bounds
alone would accept an all-zero output on the MLA config)."""
import numpy as np
import pytest

import oracle
import workloads as W
from workloads import KIND_KV, KIND_MLA, ModelCfg

pytestmark = pytest.mark.gpu

MAX_ABS, MEAN_ABS, LSE_ABS, REL_FRO = 1e-2, 1e-3, 1e-3, 1e-2


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device (no CPU fallback exists)"
    return torch


def device_workload(w, **kw):
    from paper_2606_24506_b200.harness import DeviceWorkload
    return DeviceWorkload(w, **kw)


def compare(w, got, ref, label=""):
    """got/ref: lists of (O, LSE) per request."""
    all_abs = []
    worst = {"max_abs": 0.0, "lse": 0.0, "rel": 0.0}
    for i, ((o, l), (ro, rl)) in enumerate(zip(got, ref)):
        assert np.isfinite(o).all() and np.isfinite(l).all(), "%s request %d: non-finite output" % (label, i)
        d = np.abs(o.astype(np.float64) - ro)
        all_abs.append(d.reshape(-1))
        rel = np.linalg.norm(o.astype(np.float64) - ro) / np.linalg.norm(ro)
        worst["max_abs"] = max(worst["max_abs"], d.max())
        worst["lse"] = max(worst["lse"], np.abs(l.astype(np.float64) - rl).max())
        worst["rel"] = max(worst["rel"], rel)
        assert rel <= REL_FRO, "%s request %d: relative error %.3e" % (label, i, rel)
    mean_abs = np.concatenate(all_abs).mean()
    assert worst["max_abs"] <= MAX_ABS, (label, worst)
    assert mean_abs <= MEAN_ABS, (label, mean_abs)
    assert worst["lse"] <= LSE_ABS, (label, worst)
    worst["mean_abs"] = mean_abs
    return worst


def run_and_compare(w, label="", options=None, heads=None):
    dw = device_workload(w)
    try:
        for k, v in (options or {}).items():
            dw.pool.set_option(k, v)
        dw.out.fill_(float("nan"))
        dw.lse.fill_(float("nan"))
        dw.ensure_workspace()
        dw.ws.fill_(0xFF)            # split partials start as NaN: a combine that reads one too early shows
        dw.decode()
        got = dw.results()
        # a second launch on the same pool must give the same bits (counters reset, determinism); the
        # workspace is poisoned again, so partials left by the first launch cannot stand in for late ones
        dw.out.fill_(float("nan"))
        dw.ws.fill_(0xFF)
        dw.decode()
        got2 = dw.results()
        for (o, l), (o2, l2) in zip(got, got2):
            assert np.array_equal(o, o2) and np.array_equal(l, l2), "%s: relaunch differs" % label
    finally:
        dw.close()
    ref = oracle.decode_workload(w)
    return compare(w, got, ref, label)


# ------------------------------------------------------------------ gather: bit-exact
@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_gather_bit_exact_all_configs(torch_cuda, k):
    w = W.config(k)
    dw = device_workload(w)
    try:
        # cfg5 has 64 requests: check them all (the copies are cheap)
        for i, r in enumerate(w.requests):
            m = w.models[r.model_id]
            gk, gv = dw.gather(i)
            rk, rv = oracle.gather(w.arena, w.page_tokens, w.page_bytes, w.num_pages, m.kind,
                                   m.n_kv_heads, m.head_dim_qk, m.head_dim_v, r.page_ids, r.context_len)
            assert gk.tobytes() == rk.tobytes(), "cfg%d request %d K" % (k, i)
            assert gv.tobytes() == rv.tobytes(), "cfg%d request %d V" % (k, i)
    finally:
        dw.close()


def test_gather_arbitrary_bit_patterns(torch_cuda):
    m = ModelCfg(KIND_KV, 4, 2, 16, 8, 1.0)
    w = W.small_workload([m], [0, 0], [77, 3], page_tokens=8, seed=5)
    rng = np.random.default_rng(6)
    w.arena[:] = rng.integers(0, 65536, size=w.arena.size).astype(np.uint16)   # NaNs, -0, denormals
    dw = device_workload(w)
    try:
        for i, r in enumerate(w.requests):
            gk, gv = dw.gather(i)
            rk, rv = oracle.gather(w.arena, 8, w.page_bytes, w.num_pages, 0, 2, 16, 8, r.page_ids, r.context_len)
            assert gk.tobytes() == rk.tobytes() and gv.tobytes() == rv.tobytes()
    finally:
        dw.close()


# ------------------------------------------------------------------ attention: small shapes, every kernel
SMALL = [
    # (models, req_models, req_ctx, P, value_shift)  -- several tiles and a ragged tail each
    ([ModelCfg(KIND_KV, 8, 1, 128, 128, 128 ** -0.5)], [0, 0, 0], [1, 17, 1000], 16, 0.0),
    ([ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5)], [0, 0], [4097, 700], 64, 0.0),
    ([ModelCfg(KIND_KV, 32, 1, 128, 128, 128 ** -0.5)], [0], [9999], 64, 3.0),
    ([ModelCfg(KIND_KV, 64, 8, 128, 128, 128 ** -0.5), ModelCfg(KIND_KV, 16, 1, 128, 128, 128 ** -0.5)],
     [0, 1, 1, 0, 1], [333, 5000, 31, 2049, 128], 32, 0.0),
    ([ModelCfg(KIND_KV, 12, 3, 64, 32, 0.2)], [0, 0], [500, 65], 16, 0.0),       # generic shapes
    ([ModelCfg(KIND_KV, 40, 2, 128, 128, 0.1)], [0], [3000], 128, 3.0),          # g = 20 (ragged m-tile)
    ([ModelCfg(KIND_MLA, 128, 1, 576, 512, 192 ** -0.5)], [0, 0], [2000, 129], 64, 0.0),
    ([ModelCfg(KIND_MLA, 16, 1, 576, 512, 192 ** -0.5)], [0], [777], 64, 0.0),
    ([ModelCfg(KIND_MLA, 8, 1, 64, 32, 0.3), ModelCfg(KIND_KV, 4, 2, 64, 64, 0.3)], [0, 1, 0], [100, 200, 7], 8, 0.0),
    # MHA (Hq = Hkv, group size 1; the paper's Type I models, SURVEY 8(f) N4 names the variant)
    ([ModelCfg(KIND_KV, 8, 8, 128, 128, 128 ** -0.5), ModelCfg(KIND_KV, 4, 4, 64, 64, 0.125)], [0, 1, 0], [1500, 300, 33], 16, 0.0),
]


@pytest.mark.parametrize("case", range(len(SMALL)))
@pytest.mark.parametrize("kernel", [0, 1, 2, 3])
def test_attention_small(torch_cuda, case, kernel):
    import paper_2606_24506_b200 as cp
    models, rm, rc, P, shift = SMALL[case]
    scale = 0.1 if models[0].kind == KIND_MLA and models[0].head_dim_qk == 576 else 1.0
    w = W.small_workload(models, rm, rc, page_tokens=P, seed=100 + case, value_scale=scale,
                         value_shift=shift, keep_contiguous=False)
    # few CTAs' worth of target tiles would give one tile per group: force real splitting
    worst = run_and_compare(w, "small%d/k%d" % (case, kernel),
                            {cp.CP_OPT_KERNEL: kernel, cp.CP_OPT_MIN_TILE_PAGES: 1})
    print("small case %d kernel %d: %s" % (case, kernel, worst))


def test_outputs_of_order_one_mla(torch_cuda):
    """O(1)-sized outputs on the MLA shape: one dominant key and shifted latents, so that an
    all-zero or mis-scaled result cannot hide under the absolute tolerances."""
    import paper_2606_24506_b200 as cp
    m = ModelCfg(KIND_MLA, 128, 1, 576, 512, 192 ** -0.5)
    w = W.small_workload([m], [0], [3000], page_tokens=64, seed=321, value_scale=0.1,
                         keep_contiguous=False)
    # make token 1234 dominant for every head: k = 40 * mean-direction of the queries
    q = W.bf16_to_f64(w.q[0])
    direction = q.mean(0)
    direction /= np.linalg.norm(direction)
    r = w.requests[0]
    pid = int(r.page_ids[1234 // 64])
    row = w.arena.reshape(w.num_pages, -1)[pid].reshape(64, 576)
    row[1234 % 64] = W.f32_to_bf16((direction * 6.0 + 1.0).astype(np.float32))
    for kernel in (0, 1, 2):
        worst = run_and_compare(w, "mla_O1/k%d" % kernel, {cp.CP_OPT_KERNEL: kernel})
        print(worst)


def _add_logit_ramp(w, req_index, amp, dims):
    """Make the logits of request `req_index` rise steadily along the context (by about
    sigma * 4 * amp in total): q_h += 4 u, k_t += amp (t / T) u with u a unit vector supported on
    `dims`.  The running softmax reference then has to move many times (the kernels' lazy
    reference update and, on the MLA path, the rescale of O in tensor memory)."""
    r = w.requests[req_index]
    m = w.models[r.model_id]
    P, d = w.page_tokens, m.head_dim_qk
    u = np.zeros(d)
    u[dims] = np.random.default_rng(5).standard_normal(len(dims))
    u /= np.linalg.norm(u)
    w.q[req_index] = W.f32_to_bf16((W.bf16_to_f64(w.q[req_index]) + 4.0 * u).astype(np.float32))
    pages = w.arena.reshape(w.num_pages, -1)
    n_lp = -(-r.context_len // P)
    for lp in range(n_lp):
        t = lp * P + np.arange(P)
        ramp = (amp * np.minimum(t, r.context_len - 1) / r.context_len)[:, None] * u[None, :]
        for c in range(m.n_kv_heads):
            blk = pages[int(r.page_ids[lp * m.n_kv_heads + c])][:P * d].reshape(P, d)
            valid = min(P, r.context_len - lp * P)
            k = W.bf16_to_f64(blk[:valid]) + ramp[:valid]
            blk[:valid] = W.f32_to_bf16(k.astype(np.float32))


@pytest.mark.parametrize("kind", ["kv", "mla"])
def test_rising_logits_move_the_softmax_reference(torch_cuda, kind):
    import paper_2606_24506_b200 as cp
    if kind == "kv":
        m = ModelCfg(KIND_KV, 16, 1, 128, 128, 128 ** -0.5)
        w = W.small_workload([m], [0, 0], [3000, 700], page_tokens=64, seed=11, keep_contiguous=False)
        _add_logit_ramp(w, 0, 200.0, list(range(128)))
    else:
        m = ModelCfg(KIND_MLA, 128, 1, 576, 512, 192 ** -0.5)
        w = W.small_workload([m], [0, 0], [3000, 700], page_tokens=64, seed=12, value_scale=0.1,
                             keep_contiguous=False)
        _add_logit_ramp(w, 0, 240.0, list(range(512, 576)))      # rope part only: values untouched
    ref_lse = oracle.decode_workload(w)[0][1]
    assert ref_lse.max() - ref_lse.min() >= 0 and ref_lse.max() > 30.0     # the ramp is really there
    for kernel in (0, 1, 2, 3):
        for mtp in (1, 100000):                                  # many short tiles / one tile per group
            worst = run_and_compare(w, "ramp_%s/k%d/mtp%d" % (kind, kernel, mtp),
                                    {cp.CP_OPT_KERNEL: kernel, cp.CP_OPT_MIN_TILE_PAGES: mtp})
            print(worst)


@pytest.mark.parametrize("n_ctas", [2, 4, 6])
@pytest.mark.parametrize("kernel", [0, 2, 3])
def test_few_ctas_many_tiles_per_cta(torch_cuda, n_ctas, kernel):
    """Persistent loops over many work items per CTA (or CTA pair): a grid of 2..6 CTAs on batches
    that yield dozens of tiles, with group changes in between (query restaging, ring phases across
    tiles, statically assigned combine units on a small grid)."""
    import paper_2606_24506_b200 as cp
    cases = [
        ([ModelCfg(KIND_MLA, 128, 1, 576, 512, 192 ** -0.5), ModelCfg(KIND_MLA, 48, 1, 576, 512, 192 ** -0.5)],
         [0, 1, 0], [1500, 700, 65], 64, 0.1),
        ([ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5), ModelCfg(KIND_KV, 16, 1, 128, 128, 128 ** -0.5)],
         [0, 1, 1], [1500, 3000, 65], 64, 1.0),
    ]
    for models, rm, rc, P, scale in cases:
        w = W.small_workload(models, rm, rc, page_tokens=P, seed=55, value_scale=scale, keep_contiguous=False)
        worst = run_and_compare(w, "few_ctas%d/k%d" % (n_ctas, kernel),
                                {cp.CP_OPT_KERNEL: kernel, cp.CP_OPT_NUM_CTAS: n_ctas,
                                 cp.CP_OPT_MIN_TILE_PAGES: 1, cp.CP_OPT_WAVES_X16: 16 * 12})
        print(worst)


@pytest.mark.parametrize("P", [32, 128])
def test_mla_other_page_sizes(torch_cuda, P):
    """MLA tensor-core kernels with 1 and 4 slices per page (P = 32, 128); P = 16 falls back to the
    generic kernel (slices are 32 tokens) and must still be right."""
    import paper_2606_24506_b200 as cp
    m = ModelCfg(KIND_MLA, 128, 1, 576, 512, 192 ** -0.5)
    for pt in (P, 16):
        w = W.small_workload([m], [0, 0], [1111, 97], page_tokens=pt, seed=77, value_scale=0.1, keep_contiguous=False)
        for kernel in (0, 2):
            worst = run_and_compare(w, "mla_P%d/k%d" % (pt, kernel), {cp.CP_OPT_KERNEL: kernel, cp.CP_OPT_MIN_TILE_PAGES: 1})
            print(worst)


def test_kv_and_mla_models_share_one_pool(torch_cuda):
    """GQA, MQA and MLA models colocated in ONE pool of fixed-size pages (page_bytes = the MLA page,
    73 728 B; the K/V models use the first 32 KiB of theirs): one cp_decode_attention call = one
    tensor-core launch per attention kind, pages of all models interleaved."""
    import paper_2606_24506_b200 as cp
    models = [ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5), ModelCfg(KIND_MLA, 128, 1, 576, 512, 192 ** -0.5),
              ModelCfg(KIND_KV, 16, 1, 128, 128, 128 ** -0.5)]
    w = W.small_workload(models, [0, 1, 2, 1], [700, 900, 1300, 65], page_tokens=64, seed=5, value_scale=0.3,
                         keep_contiguous=False)
    assert w.page_bytes == 64 * 576 * 2
    dw = device_workload(w)
    c0 = dw.pool.counters()["kernel_launches"]
    dw.decode()
    assert dw.pool.counters()["kernel_launches"] - c0 == 2          # one launch per kind, no per-request launches
    dw.close()
    for kernel in (0, 2):
        worst = run_and_compare(w, "mixed_kinds/k%d" % kernel, {cp.CP_OPT_KERNEL: kernel, cp.CP_OPT_MIN_TILE_PAGES: 1})
        print(worst)


# ------------------------------------------------------------------ invariants on the GPU path
def test_page_permutation_is_bit_identical(torch_cuda):
    """P5 on the GPU: split boundaries are logical, so moving the data to other physical
    pages must not change a single bit."""
    m = ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5)
    a = W.small_workload([m], [0, 0], [5000, 333], page_tokens=64, seed=7, extra_pages=5)
    b = W.small_workload([m], [0, 0], [5000, 333], page_tokens=64, seed=7, extra_pages=5)
    # b: same logical data, different physical placement
    perm = np.random.default_rng(99).permutation(b.num_pages)
    pages = b.arena.reshape(b.num_pages, -1)
    newp = np.empty_like(pages)
    newp[perm] = pages
    b.arena = newp.reshape(-1)
    for r in b.requests:
        r.page_ids = perm[r.page_ids].astype(np.int32)
    res = []
    for w in (a, b):
        dw = device_workload(w)
        dw.decode()
        res.append(dw.results())
        dw.close()
    for (o1, l1), (o2, l2) in zip(*res):
        assert np.array_equal(o1, o2) and np.array_equal(l1, l2)


def test_poison_and_batch_independence(torch_cuda):
    """P7 on the GPU: results do not depend on free pages, on the dead tail of the last page,
    nor on which other requests share the launch."""
    ms = [ModelCfg(KIND_KV, 16, 1, 128, 128, 128 ** -0.5), ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5)]
    w = W.small_workload(ms, [0, 1, 0], [1000, 2500, 77], page_tokens=32, seed=11, extra_pages=9)
    dw = device_workload(w)
    dw.decode()
    full = dw.results()
    dw.close()
    # rewrite everything that is not a mapped valid slot with other garbage (inf, big, NaN)
    w2 = W.small_workload(ms, [0, 1, 0], [1000, 2500, 77], page_tokens=32, seed=11, extra_pages=9)
    mask = (w2.arena == W.BF16_NAN)
    junk = np.random.default_rng(3).choice(np.array([0x7F80, 0xFF80, 0x7F7F, 0x7FFF, 0x4000], np.uint16),
                                           size=w2.arena.size)
    w2.arena[mask] = junk[mask]
    dw = device_workload(w2)
    dw.decode()
    junked = dw.results()
    # request 1 alone, and the batch in another order
    import torch
    ids = np.array([1], dtype=np.int32)
    m1 = ms[1]
    q1 = torch.from_numpy(w2.q[1].view(np.int16).reshape(-1)).cuda()
    o1 = torch.empty(m1.n_q_heads * m1.head_dim_v, dtype=torch.float32, device="cuda")
    l1 = torch.empty(m1.n_q_heads, dtype=torch.float32, device="cuda")
    dw.decode(ids=ids, q=q1, out=o1, lse=l1)
    torch.cuda.synchronize()
    alone = o1.cpu().numpy().reshape(m1.n_q_heads, m1.head_dim_v)
    dw.close()
    for (a, la), (b, lb) in zip(full, junked):
        assert np.array_equal(a, b) and np.array_equal(la, lb)
    ref = oracle.decode_workload(w2, request_indices=[1])[0]
    assert np.abs(alone - ref[0]).max() <= MAX_ABS
    assert np.linalg.norm(alone - ref[0]) / np.linalg.norm(ref[0]) <= REL_FRO


def test_golden_g1_on_gpu(torch_cuda):
    """The golden vector G1 (tests/golden/g1_kv.txt) through the CUDA path (d = 8)."""
    from test_oracle_pins import _g1_inputs, manual_workload, parse_golden, bf16
    Q, K, V = _g1_inputs()
    m = ModelCfg(KIND_KV, 2, 1, 8, 8, 1.0 / np.sqrt(8.0))
    w = manual_workload(m, 2, bf16(Q), bf16(K).reshape(5, 1, 8), bf16(V).reshape(5, 1, 8))
    dw = device_workload(w)
    dw.decode()
    (o, l), = dw.results()
    dw.close()
    g = parse_golden("g1_kv.txt")
    assert np.abs(l - g["lse"]).max() < 1e-5
    for h in range(2):
        assert np.abs(o[h] - g["out"][h]).max() < 5e-3   # P is rounded to bf16 on the tensor path


def test_append_and_context_growth(torch_cuda):
    """Decode, grow the context (same page, then a new page), decode again: the plan cache and
    the device tables follow (slow path a0), results track the oracle at every step."""
    m = ModelCfg(KIND_KV, 8, 1, 128, 128, 128 ** -0.5)
    full = W.small_workload([m], [0], [200], page_tokens=16, seed=21)
    r = full.requests[0]
    dw = device_workload(full, map_requests=False)
    n0 = 10                                     # pages mapped first: 160 tokens of capacity
    dw.pool.map_pages(0, 0, r.page_ids[:n0], 150)
    for ctx, extra in ((150, 0), (151, 0), (160, 0), (161, 1), (200, 2)):
        if extra:
            have = dw.pool.request_info(0)[2].size
            dw.pool.map_pages(0, 0, r.page_ids[have:have + extra], ctx)
        else:
            dw.pool.map_pages(0, 0, None, ctx)
        dw.decode()
        (o, l), = dw.results()
        ro, rl = oracle.attention(full.arena, 16, full.page_bytes, full.num_pages, 0, 8, 1, 128, 128,
                                  m.softmax_scale, r.page_ids, ctx, full.q[0])
        assert np.abs(o - ro).max() <= MAX_ABS and np.abs(l - rl).max() <= LSE_ABS
        assert np.linalg.norm(o - ro) / np.linalg.norm(ro) <= REL_FRO
    dw.close()


@pytest.mark.parametrize("kind", ["kv", "mla"])
def test_append_kv_matches_oracle_bit_for_bit(torch_cuda, kind):
    """cp_pool_append_kv writes one token per request per call (pages taken from the
    free list when a position opens a new logical page).  After every call the WHOLE device arena
    equals the host arena the oracle's append produced with the same page ids (bit-exact, poison
    included), and attention on the grown contexts tracks the oracle."""
    import torch
    if kind == "kv":
        models = [ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5), ModelCfg(KIND_KV, 16, 1, 128, 128, 128 ** -0.5)]
        rm, rc, P, scale = [0, 1, 1], [30, 64, 5], 16, 1.0
    else:
        models = [ModelCfg(KIND_MLA, 128, 1, 576, 512, 192 ** -0.5)]
        rm, rc, P, scale = [0, 0], [63, 130], 32, 0.1
    w = W.small_workload(models, rm, rc, page_tokens=P, seed=91, value_scale=scale, extra_pages=40,
                         keep_contiguous=False)
    dw = device_workload(w, page_list_slack=3 * max(m.n_kv_heads for m in models))
    rng = np.random.default_rng(17)
    host = w.arena.copy()
    ctx = [r.context_len for r in w.requests]
    for step in range(2 * P + 3):                       # crosses at least two page boundaries per request
        ks, vs = [], []
        for r in w.requests:
            m = models[r.model_id]
            ks.append(W.f32_to_bf16((scale * rng.standard_normal((m.n_kv_heads, m.head_dim_qk))).astype(np.float32)))
            if m.kind == KIND_KV:
                vs.append(W.f32_to_bf16((scale * rng.standard_normal((m.n_kv_heads, m.head_dim_v))).astype(np.float32)))
        k_dev = torch.from_numpy(np.concatenate([x.reshape(-1) for x in ks]).view(np.int16)).to(dw.device)
        v_dev = torch.from_numpy(np.concatenate([x.reshape(-1) for x in vs]).view(np.int16)).to(dw.device) if vs else None
        dw.pool.append_kv(dw.ids, k_dev, v_dev, dw.stream())
        vi = 0
        for i, r in enumerate(w.requests):
            m = models[r.model_id]
            _, c, ids = dw.pool.request_info(r.request_id)
            assert c == ctx[i] + 1
            r.page_ids = ids                              # the library chose the new pages
            v_new = None
            if m.kind == KIND_KV:
                v_new = vs[vi]; vi += 1
            oracle.append(host, P, w.page_bytes, w.num_pages, m.kind, m.n_kv_heads, m.head_dim_qk, m.head_dim_v,
                          ids, ctx[i], ks[i], v_new)
            ctx[i] += 1
            r.context_len = ctx[i]
        if step % P in (0, 1) or step == 2 * P + 2:
            torch.cuda.synchronize()
            assert dw.arena.cpu().numpy().view(np.uint16).tobytes() == host.tobytes(), "arena differs at step %d" % step
    w.arena = host
    dw.decode()
    got = dw.results()
    dw.close()
    worst = compare(w, got, oracle.decode_workload(w), "append_" + kind)
    print(worst)


@pytest.mark.parametrize("kind", ["kv", "kv_vmm", "mla", "mixed", "kv_warp_mma"])
def test_decode_step_appends_and_attends_in_one_call(torch_cuda, kind):
    """SURVEY 8(f) N1, second half: cp_decode_step = append + attend.  For MQA / GQA models on the tcgen05 kernel
    the iteration is ONE launch (the tile that holds a group's last page writes the new rows before requesting
    the page); other kinds / kernels get the append kernel in front.  After every step the whole device arena is
    bit-identical to the oracle's append, and the attention over the T + 1 tokens is within the bars."""
    import torch
    import paper_2606_24506_b200 as cp
    vmm = kind == "kv_vmm"
    if kind in ("kv", "kv_vmm", "kv_warp_mma"):
        models = [ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5), ModelCfg(KIND_KV, 16, 1, 128, 128, 128 ** -0.5)]
        rm, rc, P, scale = [0, 1, 1], [2500, 64, 5], 16, 1.0
    elif kind == "mla":
        models = [ModelCfg(KIND_MLA, 128, 1, 576, 512, 192 ** -0.5)]
        rm, rc, P, scale = [0, 0], [63, 700], 32, 0.1
    else:
        models = [ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5), ModelCfg(KIND_MLA, 128, 1, 576, 512, 192 ** -0.5)]
        rm, rc, P, scale = [0, 1, 0], [700, 130, 31], 32, 0.3
    w = W.small_workload(models, rm, rc, page_tokens=P, seed=93, value_scale=scale, extra_pages=60, keep_contiguous=False)
    dw = device_workload(w, page_list_slack=3 * max(m.n_kv_heads for m in models), vmm=vmm,
                         **({"vmm_budget_bytes": (w.num_pages + 64) * w.page_bytes + (16 << 20)} if vmm else {}))
    dw.pool.set_option(cp.CP_OPT_MIN_TILE_PAGES, 1)
    if kind == "kv_warp_mma":
        dw.pool.set_option(cp.CP_OPT_KERNEL, 3)
    rng = np.random.default_rng(19)
    host = w.arena.copy()
    ctx = [r.context_len for r in w.requests]
    host_free = sorted(set(range(w.num_pages)) - set(int(x) for r in w.requests for x in r.page_ids))
    n_steps = 2 * P + 3
    for step in range(n_steps):                       # crosses at least two page boundaries per request
        ks, vs, qs = [], [], []
        for r in w.requests:
            m = models[r.model_id]
            ks.append(W.f32_to_bf16((scale * rng.standard_normal((m.n_kv_heads, m.head_dim_qk))).astype(np.float32)))
            if m.kind == KIND_KV:
                vs.append(W.f32_to_bf16((scale * rng.standard_normal((m.n_kv_heads, m.head_dim_v))).astype(np.float32)))
            qs.append(W.f32_to_bf16((scale * rng.standard_normal((m.n_q_heads, m.head_dim_qk))).astype(np.float32)))
        k_dev = torch.from_numpy(np.concatenate([x.reshape(-1) for x in ks]).view(np.int16)).to(dw.device)
        v_dev = torch.from_numpy(np.concatenate([x.reshape(-1) for x in vs]).view(np.int16)).to(dw.device) if vs else None
        q_dev = torch.from_numpy(np.concatenate([x.reshape(-1) for x in qs]).view(np.int16)).to(dw.device)
        need = max(dw.pool.decode_step_workspace_bytes(dw.ids), 256)
        ws = torch.full((need,), 0xFF, dtype=torch.uint8, device=dw.device)
        dw.out.fill_(float("nan"))
        dw.lse.fill_(float("nan"))
        c0 = dw.pool.counters()["kernel_launches"]
        dw.pool.decode_step(dw.ids, k_dev, v_dev, q_dev, dw.out, dw.lse, ws, need, dw.stream())
        launches = dw.pool.counters()["kernel_launches"] - c0
        if kind in ("kv", "kv_vmm"):
            assert launches == 1, "the fused iteration must be one launch, got %d" % launches
        elif kind == "mixed":
            assert launches == 3          # append kernel for the MLA requests, then one decode launch per kind
        vi = 0
        for i, r in enumerate(w.requests):
            m = models[r.model_id]
            _, c, ids = dw.pool.request_info(r.request_id)
            assert c == ctx[i] + 1
            v_new = None
            if m.kind == KIND_KV:
                v_new = vs[vi]; vi += 1
            if vmm:
                # the library's arena is its own contiguous virtual range: the oracle keeps the host image and takes
                # pages of its own choice when a position opens one (where a page lies does not enter the results)
                if ctx[i] % P == 0 and ctx[i] // P * m.n_kv_heads >= r.page_ids.size:
                    r.page_ids = np.concatenate([r.page_ids, np.array([host_free.pop() for _ in range(m.n_kv_heads)], dtype=np.int32)])
            else:
                r.page_ids = ids
            oracle.append(host, P, w.page_bytes, w.num_pages, m.kind, m.n_kv_heads, m.head_dim_qk, m.head_dim_v,
                          r.page_ids, ctx[i], ks[i], v_new)
            ctx[i] += 1
            r.context_len = ctx[i]
            w.q[i] = qs[i]
        if step % P in (0, 1, 2) or step == n_steps - 1:
            torch.cuda.synchronize()
            if not vmm:
                assert dw.arena.cpu().numpy().view(np.uint16).tobytes() == host.tobytes(), "arena differs at step %d" % step
            w.arena = host
            got = dw.results()
            worst = compare(w, got, oracle.decode_workload(w), "decode_step_%s_%d" % (kind, step))
    print(worst)
    # too small a workspace: the append is taken back, nothing changed
    before = [dw.pool.request_info(r.request_id) for r in w.requests]
    free_before = dw.pool.stats()
    if dw.pool.decode_step_workspace_bytes(dw.ids) > 0:
        with pytest.raises(cp.CrossPoolError) as e:
            dw.pool.decode_step(dw.ids, k_dev, v_dev, q_dev, dw.out, dw.lse, ws, 16, dw.stream())
        assert e.value.status == cp.CP_ERR_WORKSPACE
        after = [dw.pool.request_info(r.request_id) for r in w.requests]
        assert all(a[1] == b[1] and list(a[2]) == list(b[2]) for a, b in zip(after, before)) and dw.pool.stats() == free_before
    dw.close()


def test_mixed_kinds_run_side_by_side(torch_cuda):
    """A batch with MQA/GQA and MLA models: one launch per kind, on two streams, so that the second kernel's CTAs
    move in as the first one's leave (its tail and the other's start-up overlap): the step takes less than the two
    kinds take one after the other.  (Splitting the SMs between the kinds was measured and is slower: each kernel
    needs every SM to reach its own rate.)"""
    torch = torch_cuda
    models = [ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5), ModelCfg(KIND_MLA, 128, 1, 576, 512, 192 ** -0.5)]
    w = W.small_workload(models, [0, 1, 0, 1], [60000, 50000, 50000, 40000], page_tokens=64, seed=8, value_scale=0.3,
                         keep_contiguous=False)
    dw = device_workload(w)
    try:
        def timed(ids):
            ids = np.array(ids, dtype=np.int32)
            q = torch.from_numpy(np.concatenate([w.q[i].reshape(-1) for i in ids]).view(np.int16)).to(dw.device)
            need = max(dw.pool.decode_workspace_bytes(ids), 256)
            ws = torch.empty(need, dtype=torch.uint8, device=dw.device)
            ts = []
            for _ in range(8):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                dw.pool.decode_attention(ids, q, dw.out, dw.lse, ws, need, dw.stream())
                e1.record()
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            return float(np.median(ts[2:]))
        c0 = dw.pool.counters()["kernel_launches"]
        both = timed([0, 1, 2, 3])
        assert (dw.pool.counters()["kernel_launches"] - c0) == 2 * 8
        kv, mla = timed([0, 2]), timed([1, 3])
        print("mixed step %.1f us, K/V alone %.1f us, MLA alone %.1f us" % (1e3 * both, 1e3 * kv, 1e3 * mla))
        assert both < 0.99 * (kv + mla)
    finally:
        dw.close()
    run_and_compare(w, "mixed_side_by_side")


def test_calls_on_two_streams_are_ordered_by_the_library(torch_cuda):
    """One pool driven from two streams in turn (the paper's two in-flight batches): the work list, counters
    and tables of a plan are reused from call to call, so a call on another stream than the previous one must
    wait for it.  Each call's batch differs from the previous one's (plan rebuilt and re-uploaded while the
    other stream's kernel may still run); results must match the single-stream run bit for bit."""
    torch = torch_cuda
    import paper_2606_24506_b200 as cp
    models = [ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5), ModelCfg(KIND_KV, 16, 1, 128, 128, 128 ** -0.5)]
    w = W.small_workload(models, [0, 1, 1, 0], [40000, 90000, 3000, 25000], page_tokens=64, seed=61, keep_contiguous=False)
    dw = device_workload(w)
    dw.pool.set_option(cp.CP_OPT_MIN_TILE_PAGES, 1)
    batches = [[0, 1], [2, 3], [1, 3], [0, 2, 3], [1]]
    rows = {i: w.models[r.model_id].n_q_heads for i, r in enumerate(w.requests)}

    def run(streams):
        outs = []
        ws = torch.full((32 << 20,), 0xFF, dtype=torch.uint8, device=dw.device)
        for it in range(3):
            for bi, b in enumerate(batches):
                ids = np.array(b, dtype=np.int32)
                q = torch.from_numpy(np.concatenate([w.q[i].reshape(-1) for i in b]).view(np.int16)).to(dw.device)
                n = sum(rows[i] for i in b)
                out = torch.full((n * 128,), float("nan"), dtype=torch.float32, device=dw.device)
                lse = torch.full((n,), float("nan"), dtype=torch.float32, device=dw.device)
                torch.cuda.synchronize()
                st = streams[(it * len(batches) + bi) % len(streams)]
                dw.pool.decode_attention(ids, q, out, lse, ws, ws.numel(), st.cuda_stream)
                outs.append((out, lse))
        torch.cuda.synchronize()
        return [(o.cpu().numpy(), l.cpu().numpy()) for o, l in outs]

    try:
        s1, s2 = torch.cuda.Stream(device=dw.device), torch.cuda.Stream(device=dw.device)
        ref = run([s1])
        got = run([s1, s2])
        for i, ((o, l), (ro, rl)) in enumerate(zip(got, ref)):
            assert np.isfinite(o).all() and np.array_equal(o, ro) and np.array_equal(l, rl), "call %d differs" % i
    finally:
        dw.close()


def test_full_config4_with_order_one_outputs(torch_cuda):
    """cfg4 (batch 1, 262 144 tokens, g = 32) with V = N(0, 1) + 3: outputs are O(1) instead of ~2.5e-3, so the
    absolute bars bite as hard as the relative one (tolerance strength)."""
    w = W.config(4)
    r = w.requests[0]
    m = w.models[r.model_id]
    P, rows = w.page_tokens, w.page_bytes // 256
    arena = w.arena.reshape(w.num_pages, rows, 128)
    rng = np.random.default_rng(404)
    for lp, pid in enumerate(r.page_ids):
        n_valid = min(P, r.context_len - lp * P)
        arena[pid, P:P + n_valid, :] = W.f32_to_bf16((rng.standard_normal((n_valid, 128)) + 3.0).astype(np.float32))
    worst = run_and_compare(w, "cfg4-V+3")
    print("cfg4 with V + 3: %s" % worst)


def test_host_buffer_entry_point_matches_device_path(torch_cuda):
    torch = torch_cuda
    ms = [ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5), ModelCfg(KIND_KV, 16, 1, 128, 128, 128 ** -0.5)]
    w = W.small_workload(ms, [0, 1], [3000, 900], page_tokens=64, seed=31)
    dw = device_workload(w)
    dw.decode()
    dev = dw.results()
    need = dw.pool.decode_workspace_bytes_host(dw.ids)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    q_host = torch.from_numpy(w.q_packed().view(np.int16)).pin_memory()
    o_host = torch.empty(dw.out.numel(), dtype=torch.float32).pin_memory()
    l_host = torch.empty(dw.lse.numel(), dtype=torch.float32).pin_memory()
    dw.pool.decode_attention_host(dw.ids, q_host, o_host, l_host, ws, need, dw.stream())
    o = np.concatenate([x[0].reshape(-1) for x in dev])
    l = np.concatenate([x[1].reshape(-1) for x in dev])
    assert np.array_equal(o_host.numpy(), o) and np.array_equal(l_host.numpy(), l)
    # adjacent host buffers (LSE directly after O): the one-copy path gives the same bytes
    ol = torch.full((dw.out.numel() + dw.lse.numel() + 8,), float("nan"), dtype=torch.float32).pin_memory()
    dw.pool.decode_attention_host(dw.ids, q_host, ol[:dw.out.numel()], ol[dw.out.numel():], ws, need, dw.stream())
    assert np.array_equal(ol[:dw.out.numel()].numpy(), o)
    assert np.array_equal(ol[dw.out.numel():dw.out.numel() + dw.lse.numel()].numpy(), l)
    assert np.isnan(ol[dw.out.numel() + dw.lse.numel():].numpy()).all()          # nothing written past the end
    # the same with the in-place access of pinned buffers switched off, and with pageable host memory
    import paper_2606_24506_b200 as cp
    for zero_copy, pinned in ((0, True), (1, False), (1, True)):
        dw.pool.set_option(cp.CP_OPT_HOST_ZERO_COPY, zero_copy)
        oh = torch.full((dw.out.numel(),), float("nan"), dtype=torch.float32)
        lh = torch.full((dw.lse.numel(),), float("nan"), dtype=torch.float32)
        qh = torch.from_numpy(w.q_packed().view(np.int16).copy())
        if pinned:
            oh, lh, qh = oh.pin_memory(), lh.pin_memory(), qh.pin_memory()
        dw.pool.decode_attention_host(dw.ids, qh, oh, lh, ws, need, dw.stream())
        assert np.array_equal(oh.numpy(), o) and np.array_equal(lh.numpy(), l), (zero_copy, pinned)
    dw.close()


def test_workspace_too_small_is_rejected(torch_cuda):
    import paper_2606_24506_b200 as cp
    m = ModelCfg(KIND_KV, 8, 1, 128, 128, 128 ** -0.5)
    w = W.small_workload([m], [0], [4000], page_tokens=16, seed=41)
    dw = device_workload(w)
    need = dw.ensure_workspace()
    assert need > 0
    with pytest.raises(cp.CrossPoolError) as e:
        dw.pool.decode_attention(dw.ids, dw.q, dw.out, dw.lse, dw.ws, need - 4, dw.stream())
    assert e.value.status == cp.CP_ERR_WORKSPACE
    dw.close()


# ------------------------------------------------------------------ the five BASELINE configs, full size
@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_attention_full_config(torch_cuda, k):
    """Full-size parity in the launch configuration bench.py times (default options)."""
    w = W.config(k)
    worst = run_and_compare(w, "cfg%d" % k)
    print("cfg%d: %s" % (k, worst))


@pytest.mark.parametrize("k", [2, 3])
def test_attention_full_config_generic_kernel(torch_cuda, k):
    """The shape-generic kernel on full-size inputs (independent GPU cross-check)."""
    import paper_2606_24506_b200 as cp
    w = W.config(k) if k == 2 else W.config3(ctx=(16384, 4096))
    worst = run_and_compare(w, "cfg%d-generic" % k, {cp.CP_OPT_KERNEL: 1})
    print("cfg%d generic: %s" % (k, worst))


@pytest.mark.parametrize("k", [2, 4, 5])
def test_attention_full_config_warp_mma_kernel(torch_cuda, k):
    """The warp-MMA (mma.sync) K/V kernel of round 1 on full-size inputs (CP_OPT_KERNEL = 3): kept as the kernel of
    the multi-stage and q_len > 1 launches and as a second tensor-core cross-check of the tcgen05 kernel."""
    import paper_2606_24506_b200 as cp
    worst = run_and_compare(W.config(k), "cfg%d-warp-mma" % k, {cp.CP_OPT_KERNEL: 3})
    print("cfg%d warp-MMA kernel: %s" % (k, worst))


@pytest.mark.parametrize("k", [2, 4, 5])
@pytest.mark.parametrize("pct,tail,waves", [(85, 2, 16), (60, 1, 16), (0, 3, 16), (100, 2, 40)])
def test_attention_full_config_dynamic_tail(torch_cuda, k, pct, tail, waves):
    """Full-size inputs with part of every group left to the dynamically popped tail tiles (CP_OPT_STATIC_PCT,
    CP_OPT_TAIL_TILE_SLICES) and with several static rounds per CTA: results within the same bars, and -- since
    every tile is a fixed token range with its own split slot -- identical bits on a relaunch whatever CTA ran it."""
    import paper_2606_24506_b200 as cp
    worst = run_and_compare(W.config(k), "cfg%d-tail%d/%d/%d" % (k, pct, tail, waves),
                            {cp.CP_OPT_STATIC_PCT: pct, cp.CP_OPT_TAIL_TILE_SLICES: tail, cp.CP_OPT_WAVES_X16: waves})
    print("cfg%d pct %d tail %d waves %d: %s" % (k, pct, tail, waves, worst))


def test_attention_full_config_mla_single_cta_kernel(torch_cuda):
    """cfg3 at full size on the single-CTA tcgen05 MLA kernel (CP_OPT_KERNEL = 2); the default
    path (CTA pairs) is covered by test_attention_full_config."""
    import paper_2606_24506_b200 as cp
    worst = run_and_compare(W.config(3), "cfg3-single-cta", {cp.CP_OPT_KERNEL: 2})
    print("cfg3 single-CTA kernel: %s" % worst)
