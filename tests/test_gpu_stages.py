"""GPU parity of the multi-stage persistent launch (cp_decode_attention_stages, the
attention-only mock of PAPER.md §3.2/§3.3): two in-flight batches of different models and layer
counts, a third fetched when the first finishes, every layer of every batch one stage of ONE launch.
Each stage is compared with oracle.decode_stages under the bars of test_gpu_parity.py; outputs are
NaN-prefilled, so a stage that read its predecessor's output too early cannot pass."""
import numpy as np
import pytest

import oracle
import workloads as W
from workloads import KIND_KV, KIND_MLA, ModelCfg
from test_gpu_parity import LSE_ABS, MAX_ABS, MEAN_ABS, REL_FRO, device_workload, torch_cuda  # noqa: F401

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(180)]

GQA = ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5)
MQA = ModelCfg(KIND_KV, 16, 1, 128, 128, 128 ** -0.5)
MHA = ModelCfg(KIND_KV, 8, 8, 128, 128, 128 ** -0.5)


def pipeline_order(layers, slots=2):
    """Stage order of the layer-wise state machine: `slots` batches in flight, served in turn, each
    advancing its own layer cursor; a finished batch is replaced by the next one of the queue.
    Returns [(batch, layer)]."""
    queue = list(range(len(layers)))
    live = [queue.pop(0) for _ in range(min(slots, len(queue)))]
    cursor = {b: 0 for b in live}
    order = []
    while live:
        for i in range(len(live)):
            b = live[i]
            if b is None:
                continue
            order.append((b, cursor[b]))
            cursor[b] += 1
            if cursor[b] == layers[b]:
                live[i] = queue.pop(0) if queue else None
                if live[i] is not None:
                    cursor[live[i]] = 0
        live = [b for b in live if b is not None] if all(b is None for b in live) else live
    return order


def build_case(batches, P, seed):
    """batches: [(model, [context lengths], n_layers)].  One pool request per (batch, request, layer)."""
    models, rm, rc, index = [], [], [], {}
    for b, (m, ctxs, n_layers) in enumerate(batches):
        if m not in models:
            models.append(m)
        for layer in range(n_layers):
            for j, c in enumerate(ctxs):
                index[(b, layer, j)] = len(rm)
                rm.append(models.index(m))
                rc.append(c + 3 * layer)                 # the cache of a deeper layer is not a copy
    w = W.small_workload(models, rm, rc, page_tokens=P, seed=seed, keep_contiguous=False)
    order = pipeline_order([n for _, _, n in batches])
    pos = {bl: s for s, bl in enumerate(order)}
    stages = [[index[(b, layer, j)] for j in range(len(batches[b][1]))] for b, layer in order]
    deps = [pos[(b, layer - 1)] if layer > 0 else -1 for b, layer in order]
    rng = np.random.default_rng(seed + 7)
    q_in = [[W.f32_to_bf16(rng.standard_normal((w.models[w.requests[ri].model_id].n_q_heads, 128)).astype(np.float32))
             for ri in st] for st in stages]
    return w, order, stages, deps, q_in


def run_stages(torch, dw, w, stages, deps, q_in, alpha, relaunch=True):
    dev = dw.device
    ids = [[w.requests[ri].request_id for ri in st] for st in stages]
    q = torch.from_numpy(np.concatenate([x.reshape(-1) for st in q_in for x in st]).view(np.int16)).to(dev)
    rows = sum(x.shape[0] for st in q_in for x in st)
    out = torch.full((rows * 128,), float("nan"), dtype=torch.float32, device=dev)
    lse = torch.full((rows,), float("nan"), dtype=torch.float32, device=dev)
    wsb = max(dw.pool.decode_stages_workspace_bytes(ids, deps), 256)
    ws = torch.empty(wsb, dtype=torch.uint8, device=dev)
    dw.pool.decode_attention_stages(ids, deps, alpha, q, out, lse, ws, wsb, dw.stream())
    torch.cuda.synchronize()
    o, l = out.cpu().numpy(), lse.cpu().numpy()
    if relaunch:                                       # the other counter set, same bits
        out.fill_(float("nan"))
        dw.pool.decode_attention_stages(ids, deps, alpha, q, out, lse, ws, wsb, dw.stream())
        torch.cuda.synchronize()
        assert np.array_equal(o, out.cpu().numpy()) and np.array_equal(l, lse.cpu().numpy())
    res, ro = [], 0
    for st in q_in:
        cur = []
        for x in st:
            h = x.shape[0]
            cur.append((o[ro * 128:(ro + h) * 128].reshape(h, 128).copy(), l[ro:ro + h].copy()))
            ro += h
        res.append(cur)
    return res


# A dependent stage re-quantises its query to bf16 from the previous output, and the two sides' previous
# outputs differ within their own tolerance (1e-4 .. 1e-3): wherever that difference straddles a
# rounding boundary one query entry moves by a bf16 ulp (2^-8 relative), which moves a logit -- and for a
# short context the LSE -- by sigma * 2^-8 * |q_d| |k_d| ~ 1e-3 per flipped entry, a few entries per
# head.  The O bars stay those of north_star; the LSE bar of dependent stages is 1e-2.
LSE_ABS_DEPENDENT = 1e-2


def compare_stage(got, ref, dependent, label):
    all_abs, worst = [], {"max_abs": 0.0, "lse": 0.0, "rel": 0.0}
    for i, ((o, l), (ro, rl)) in enumerate(zip(got, ref)):
        assert np.isfinite(o).all() and np.isfinite(l).all(), "%s request %d: non-finite output" % (label, i)
        d = np.abs(o.astype(np.float64) - ro)
        all_abs.append(d.reshape(-1))
        worst["max_abs"] = max(worst["max_abs"], d.max())
        worst["lse"] = max(worst["lse"], np.abs(l.astype(np.float64) - rl).max())
        worst["rel"] = max(worst["rel"], np.linalg.norm(o.astype(np.float64) - ro) / np.linalg.norm(ro))
    worst["mean_abs"] = np.concatenate(all_abs).mean()
    assert worst["max_abs"] <= MAX_ABS and worst["mean_abs"] <= MEAN_ABS and worst["rel"] <= REL_FRO, (label, worst)
    assert worst["lse"] <= (LSE_ABS_DEPENDENT if dependent else LSE_ABS), (label, worst)
    return worst


BATCHES = [(GQA, [700, 33], 3), (MQA, [1500, 9, 260], 5), (MHA, [410], 2)]


def test_pipeline_order_is_the_papers_state_machine():
    assert pipeline_order([3, 5, 2]) == [(0, 0), (1, 0), (0, 1), (1, 1), (0, 2), (1, 2), (2, 0), (1, 3), (2, 1), (1, 4)]


@pytest.mark.parametrize("n_ctas", [0, 2, 5])
@pytest.mark.parametrize("P", [16, 64])
def test_stages_match_oracle(torch_cuda, n_ctas, P):
    import paper_2606_24506_b200 as cp
    w, order, stages, deps, q_in = build_case(BATCHES, P, seed=400 + P)
    ref = oracle.decode_stages(w, stages, deps, q_in, alpha=1.0)
    dw = device_workload(w)
    try:
        dw.pool.set_option(cp.CP_OPT_MIN_TILE_PAGES, 1)
        if n_ctas:
            dw.pool.set_option(cp.CP_OPT_NUM_CTAS, n_ctas)
        got = run_stages(torch_cuda, dw, w, stages, deps, q_in, 1.0)
    finally:
        dw.close()
    for s, (b, layer) in enumerate(order):
        worst = compare_stage(got[s], ref[s], deps[s] >= 0, "stage %d (batch %d layer %d)" % (s, b, layer))
    print("P=%d ctas=%d last stage: %s" % (P, n_ctas, worst))


def test_stages_alpha_zero_equal_single_steps_bit_for_bit(torch_cuda):
    """With alpha = 0 a dependent stage's query is q_in itself, so every stage must reproduce the
    single-step launch on the same requests exactly (same tiles, same combine order) -- while still
    going through the dependency waits."""
    import paper_2606_24506_b200 as cp
    torch = torch_cuda
    w, order, stages, deps, q_in = build_case(BATCHES, 32, seed=77)
    dw = device_workload(w)
    try:
        dw.pool.set_option(cp.CP_OPT_MIN_TILE_PAGES, 1)
        # the multi-stage launch runs on the warp-MMA K/V kernel: compare with the single step on the same kernel
        # (the default single step is the tcgen05 kernel, whose tiling and summation order differ)
        dw.pool.set_option(cp.CP_OPT_KERNEL, 3)
        got = run_stages(torch, dw, w, stages, deps, q_in, 0.0)
        for s, st in enumerate(stages):
            ids = np.array([w.requests[ri].request_id for ri in st], dtype=np.int32)
            q = torch.from_numpy(np.concatenate([x.reshape(-1) for x in q_in[s]]).view(np.int16)).to(dw.device)
            rows = sum(x.shape[0] for x in q_in[s])
            out = torch.full((rows * 128,), float("nan"), dtype=torch.float32, device=dw.device)
            lse = torch.full((rows,), float("nan"), dtype=torch.float32, device=dw.device)
            dw.decode(ids=ids, q=q, out=out, lse=lse)
            torch.cuda.synchronize()
            o = np.concatenate([x[0].reshape(-1) for x in got[s]])
            l = np.concatenate([x[1] for x in got[s]])
            assert np.array_equal(o, out.cpu().numpy()) and np.array_equal(l, lse.cpu().numpy()), "stage %d" % s
    finally:
        dw.close()


def teacher_forced_reference(w, stages, deps, q_in, alpha, got):
    """Oracle stage s fed the GPU's OWN output of stage deps[s]: both sides then quantise the same previous
    output, the bf16 rounding of the query cannot differ, and the dependent stage is held to the plain bars
    (LSE 1e-3) -- a real 5e-3 LSE error in a dependent stage cannot hide behind the free-running 1e-2."""
    ref = []
    for s, reqs in enumerate(stages):
        res = []
        for j, ri in enumerate(reqs):
            r = w.requests[ri]
            m = w.models[r.model_id]
            q = np.ascontiguousarray(q_in[s][j], dtype=np.uint16)
            if deps[s] >= 0:
                q = oracle.stage_query(q, got[deps[s]][j][0], alpha)
            res.append(oracle.attention(w.arena, w.page_tokens, w.page_bytes, w.num_pages, m.kind, m.n_q_heads,
                                        m.n_kv_heads, m.head_dim_qk, m.head_dim_v, m.softmax_scale, r.page_ids,
                                        r.context_len, q))
        ref.append(res)
    return ref


@pytest.mark.parametrize("P", [16, 64])
def test_dependent_stages_teacher_forced_at_the_plain_lse_bar(torch_cuda, P):
    import paper_2606_24506_b200 as cp
    w, order, stages, deps, q_in = build_case(BATCHES, P, seed=410 + P)
    dw = device_workload(w)
    try:
        dw.pool.set_option(cp.CP_OPT_MIN_TILE_PAGES, 1)
        got = run_stages(torch_cuda, dw, w, stages, deps, q_in, 1.0)
    finally:
        dw.close()
    ref = teacher_forced_reference(w, stages, deps, q_in, 1.0, got)
    for s, (b, layer) in enumerate(order):
        worst = compare_stage(got[s], ref[s], False, "teacher-forced stage %d (batch %d layer %d)" % (s, b, layer))
    print("P=%d teacher-forced, last stage: %s" % (P, worst))


def test_stages_argument_errors(torch_cuda):
    import paper_2606_24506_b200 as cp
    torch = torch_cuda
    mla = ModelCfg(KIND_MLA, 16, 1, 576, 512, 0.07)
    w = W.small_workload([GQA, MQA, mla], [0, 0, 1, 2], [100, 50, 60, 64], page_tokens=64, seed=3,
                         keep_contiguous=False, value_scale=0.1)
    dw = device_workload(w)
    try:
        buf = torch.zeros(1 << 20, dtype=torch.float32, device=dw.device)
        def call(stages, deps, alpha=1.0):
            dw.pool.decode_attention_stages(stages, deps, alpha, buf, buf, buf, buf, buf.numel() * 4, dw.stream())
        for stages, deps, status in (([[0], [1]], [-1, 1], cp.CP_ERR_INVALID_ARG),        # depends on itself
                                     ([[0, 1], [0]], [-1, 0], cp.CP_ERR_INVALID_ARG),     # other batch size
                                     ([[0], [2]], [-1, 0], cp.CP_ERR_INVALID_ARG),        # other model
                                     ([[0, 0]], [-1], cp.CP_ERR_INVALID_ARG),             # id twice in a stage
                                     ([[3]], [-1], cp.CP_ERR_UNSUPPORTED)):               # MLA
            with pytest.raises(cp.CrossPoolError) as e:
                call(stages, deps)
            assert e.value.status == status, (stages, deps)
        with pytest.raises(cp.CrossPoolError) as e:
            call([[0], [1]], [-1, 0], float("nan"))
        assert e.value.status == cp.CP_ERR_INVALID_ARG
        call([[0], [1], [0]], [-1, 0, 1])              # ids may repeat across stages
        torch.cuda.synchronize()
    finally:
        dw.close()


def test_gated_launch_follows_the_hosts_admissions(torch_cuda):
    """The doorbell variant: the kernel is launched with two stages admitted, the host admits the rest
    in two steps from another stream while the kernel is running.  The launch cannot finish before
    the last admission, finishes right after it, and computes the same bits as the ungated launch."""
    import time
    import paper_2606_24506_b200 as cp
    torch = torch_cuda
    w, order, stages, deps, q_in = build_case(BATCHES, 32, seed=123)
    dw = device_workload(w)
    try:
        dw.pool.set_option(cp.CP_OPT_MIN_TILE_PAGES, 1)
        base = run_stages(torch, dw, w, stages, deps, q_in, 1.0, relaunch=False)
        dev = dw.device
        ids = [[w.requests[ri].request_id for ri in st] for st in stages]
        q = torch.from_numpy(np.concatenate([x.reshape(-1) for st in q_in for x in st]).view(np.int16)).to(dev)
        rows = sum(x.shape[0] for st in q_in for x in st)
        out = torch.full((rows * 128,), float("nan"), dtype=torch.float32, device=dev)
        lse = torch.full((rows,), float("nan"), dtype=torch.float32, device=dev)
        wsb = max(dw.pool.decode_stages_workspace_bytes(ids, deps), 256)
        ws = torch.empty(wsb, dtype=torch.uint8, device=dev)
        published = torch.tensor([2], dtype=torch.int32, device=dev)
        steps = [torch.tensor([v], dtype=torch.int32).pin_memory() for v in (5, len(stages))]
        run, side = torch.cuda.Stream(), torch.cuda.Stream()
        torch.cuda.synchronize()
        done = torch.cuda.Event()
        t0 = time.perf_counter()
        dw.pool.decode_attention_stages_gated(ids, deps, 1.0, q, out, lse, ws, wsb, run.cuda_stream, published, 5000)
        done.record(run)
        with torch.cuda.stream(side):
            time.sleep(0.02)
            assert not done.query(), "the launch finished before all its stages were admitted"
            published.copy_(steps[0], non_blocking=True)
            side.synchronize()
            time.sleep(0.02)
            assert not done.query()
            published.copy_(steps[1], non_blocking=True)
            side.synchronize()
        run.synchronize()
        elapsed = time.perf_counter() - t0
        assert 0.04 <= elapsed < 1.0, elapsed
        assert dw.pool.decode_stages_gate_status(run.cuda_stream) == 0
        o, l = out.cpu().numpy(), lse.cpu().numpy()
        assert np.array_equal(o, np.concatenate([x[0].reshape(-1) for st in base for x in st]))
        assert np.array_equal(l, np.concatenate([x[1] for st in base for x in st]))
    finally:
        dw.close()


def test_gated_launch_times_out_instead_of_hanging(torch_cuda):
    """A doorbell the host never rings: after timeout_ms the CTAs stop gating, the launch completes with
    the right result and the status call reports the timeout."""
    import paper_2606_24506_b200 as cp
    torch = torch_cuda
    w, order, stages, deps, q_in = build_case(BATCHES[:2], 16, seed=5)
    dw = device_workload(w)
    try:
        base = run_stages(torch, dw, w, stages, deps, q_in, 0.5, relaunch=False)
        dev = dw.device
        ids = [[w.requests[ri].request_id for ri in st] for st in stages]
        q = torch.from_numpy(np.concatenate([x.reshape(-1) for st in q_in for x in st]).view(np.int16)).to(dev)
        rows = sum(x.shape[0] for st in q_in for x in st)
        out = torch.full((rows * 128,), float("nan"), dtype=torch.float32, device=dev)
        lse = torch.full((rows,), float("nan"), dtype=torch.float32, device=dev)
        wsb = max(dw.pool.decode_stages_workspace_bytes(ids, deps), 256)
        ws = torch.empty(wsb, dtype=torch.uint8, device=dev)
        published = torch.tensor([1], dtype=torch.int32, device=dev)
        dw.pool.decode_attention_stages_gated(ids, deps, 0.5, q, out, lse, ws, wsb, dw.stream(), published, 30)
        assert dw.pool.decode_stages_gate_status(dw.stream()) == 1
        assert np.array_equal(out.cpu().numpy(), np.concatenate([x[0].reshape(-1) for st in base for x in st]))
        with pytest.raises(cp.CrossPoolError) as e:
            dw.pool.decode_attention_stages_gated(ids, deps, 0.5, q, out, lse, ws, wsb, dw.stream(), published, 0)
        assert e.value.status == cp.CP_ERR_INVALID_ARG
    finally:
        dw.close()


def test_stages_on_a_vmm_arena(torch_cuda):
    """The multi-stage launch on the CUDA-VMM-backed arena (page ids by arithmetic, no table): same bits
    as on the caller-owned arena."""
    import paper_2606_24506_b200 as cp
    w, order, stages, deps, q_in = build_case(BATCHES, 64, seed=31)
    res = []
    for vmm in (False, True):
        dw = device_workload(w, vmm=vmm)
        try:
            dw.pool.set_option(cp.CP_OPT_MIN_TILE_PAGES, 1)
            res.append(run_stages(torch_cuda, dw, w, stages, deps, q_in, 1.0, relaunch=False))
        finally:
            dw.close()
    for a, b in zip(res[0], res[1]):
        for (o, l), (o2, l2) in zip(a, b):
            assert np.array_equal(o, o2) and np.array_equal(l, l2)


def test_stages_full_size_two_layers_of_cfg2(torch_cuda):
    """Full size, default options (the configuration bench.py's `stages` leg times): the eight requests of
    BASELINE cfg2 (four GQA models, 4 k - 32 k contexts) as two dependent layers, each layer with its own KV."""
    _, rm, rc = W.config2_meta()
    models = [ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5) for _ in range(4)]
    n = len(rm)
    w = W.small_workload(models, rm + rm, rc + rc, page_tokens=64, seed=2450602, keep_contiguous=False, extra_pages=64)
    stages, deps = [list(range(n)), list(range(n, 2 * n))], [-1, 0]
    rng = np.random.default_rng(11)
    q_in = [[W.f32_to_bf16(rng.standard_normal((32, 128)).astype(np.float32)) for _ in st] for st in stages]
    ref = oracle.decode_stages(w, stages, deps, q_in, alpha=1.0)
    dw = device_workload(w)
    try:
        got = run_stages(torch_cuda, dw, w, stages, deps, q_in, 1.0)
    finally:
        dw.close()
    for s in range(2):
        print("layer %d: %s" % (s, compare_stage(got[s], ref[s], deps[s] >= 0, "cfg2 layer %d" % s)))
