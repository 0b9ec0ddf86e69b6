"""GPU parity of the request queue (cp_queue_*, second half): a persistent launch that knows
nothing of its work when it starts.  The host pushes the stages of the paper's layer-wise state machine one by
one WHILE THE KERNEL RUNS (with real time between the pushes), a planner warp on the GPU cuts every batch into
tiles on arrival, and every stage must match oracle.decode_stages under the bars of test_gpu_stages.py."""
import time

import numpy as np
import pytest

import oracle
import workloads as W
from test_gpu_parity import device_workload, torch_cuda  # noqa: F401
from test_gpu_stages import BATCHES, build_case, compare_stage

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(180)]


def run_queue(torch, dw, w, stages, deps, q_in, alpha, gap_s=0.0, push_before_launch=0, close=True, timeout_ms=2000):
    import paper_2606_24506_b200 as cp
    dev = dw.device
    ids = [[w.requests[ri].request_id for ri in st] for st in stages]
    q = torch.from_numpy(np.concatenate([x.reshape(-1) for st in q_in for x in st]).view(np.int16)).to(dev)
    rows = sum(x.shape[0] for st in q_in for x in st)
    out = torch.full((rows * 128,), float("nan"), dtype=torch.float32, device=dev)
    lse = torch.full((rows,), float("nan"), dtype=torch.float32, device=dev)
    wsb = 64 << 20
    ws = torch.full((wsb,), 0xFF, dtype=torch.uint8, device=dev)
    qu = cp.Queue(dw.pool, max_stages=len(stages) + 2)
    side = torch.cuda.Stream(device=dev)               # the launch must not block the default stream's later copies
    try:
        for s in range(push_before_launch):
            assert qu.push(ids[s], deps[s], alpha) == s
        torch.cuda.synchronize()
        qu.launch(q, out, lse, ws, wsb, timeout_ms, side.cuda_stream)
        t_push = []
        for s in range(push_before_launch, len(stages)):
            if gap_s:
                time.sleep(gap_s)
            assert qu.push(ids[s], deps[s], alpha) == s
            t_push.append(time.perf_counter())
        if close:
            qu.close_queue()
        side.synchronize()
        t_done = time.perf_counter()
        st = qu.status(side.cuda_stream)
    finally:
        torch.cuda.synchronize()
        qu.free()
    o, l = out.cpu().numpy(), lse.cpu().numpy()
    res, ro = [], 0
    for stq in q_in:
        cur = []
        for x in stq:
            h = x.shape[0]
            cur.append((o[ro * 128:(ro + h) * 128].reshape(h, 128).copy(), l[ro:ro + h].copy()))
            ro += h
        res.append(cur)
    return res, st, (t_push, t_done)


@pytest.mark.parametrize("P", [16, 64])
@pytest.mark.parametrize("n_ctas", [0, 3])
def test_stages_pushed_while_the_kernel_runs_match_oracle(torch_cuda, P, n_ctas):
    import paper_2606_24506_b200 as cp
    torch = torch_cuda
    w, order, stages, deps, q_in = build_case(BATCHES, P, seed=500 + P)
    ref = oracle.decode_stages(w, stages, deps, q_in, 1.0)
    dw = device_workload(w)
    try:
        dw.pool.set_option(cp.CP_OPT_MIN_TILE_PAGES, 1)
        if n_ctas:
            dw.pool.set_option(cp.CP_OPT_NUM_CTAS, n_ctas)
        # nothing is pushed before the launch; 3 ms between pushes: the kernel idles on the queue in between
        got, st, (t_push, t_done) = run_queue(torch, dw, w, stages, deps, q_in, 1.0, gap_s=0.003)
    finally:
        dw.close()
    assert st["error"] == 0 and st["stages_planned"] == len(stages)
    assert t_done >= t_push[-1]                      # it could not have finished before the last push
    for s, (b, layer) in enumerate(order):
        worst = compare_stage(got[s], ref[s], deps[s] >= 0, "queue stage %d (batch %d layer %d)" % (s, b, layer))
    print("P=%d ctas=%d last stage: %s, planned %s" % (P, n_ctas, worst, st))


def test_queue_alpha_zero_equals_single_steps_bit_for_bit(torch_cuda):
    """alpha = 0: every queued stage must reproduce the single-step launch of the same requests on the same
    kernel (CP_OPT_KERNEL = 3) exactly -- the device-side planner cuts a batch as the host planner does."""
    import paper_2606_24506_b200 as cp
    torch = torch_cuda
    w, order, stages, deps, q_in = build_case(BATCHES, 32, seed=78)
    dw = device_workload(w)
    try:
        dw.pool.set_option(cp.CP_OPT_MIN_TILE_PAGES, 1)
        dw.pool.set_option(cp.CP_OPT_KERNEL, 3)
        got, st, _ = run_queue(torch, dw, w, stages, deps, q_in, 0.0, push_before_launch=2)
        assert st["error"] == 0
        for s, stg in enumerate(stages):
            ids = np.array([w.requests[ri].request_id for ri in stg], dtype=np.int32)
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


def test_queue_never_closed_times_out_with_what_it_has(torch_cuda):
    """A host that stops pushing without closing: the planner gives up after timeout_ms, the stages it has are
    complete and right, the error word says 1."""
    import paper_2606_24506_b200 as cp
    torch = torch_cuda
    w, order, stages, deps, q_in = build_case(BATCHES[:1], 16, seed=91)
    ref = oracle.decode_stages(w, stages, deps, q_in, 1.0)
    dw = device_workload(w)
    try:
        t0 = time.perf_counter()
        got, st, _ = run_queue(torch, dw, w, stages, deps, q_in, 1.0, close=False, timeout_ms=40)
        assert time.perf_counter() - t0 < 5.0
    finally:
        dw.close()
    assert st["error"] == 1 and st["stages_planned"] == len(stages)
    for s in range(len(stages)):
        compare_stage(got[s], ref[s], deps[s] >= 0, "queue (timed out) stage %d" % s)


def test_queue_argument_errors(torch_cuda):
    import paper_2606_24506_b200 as cp
    torch = torch_cuda
    mla = W.ModelCfg(W.KIND_MLA, 16, 1, 576, 512, 0.07)
    gqa = W.ModelCfg(W.KIND_KV, 32, 4, 128, 128, 0.09)
    w = W.small_workload([gqa, mla], [0, 1, 0], [100, 100, 50], page_tokens=64, seed=3, keep_contiguous=False)
    dw = device_workload(w)
    qu = cp.Queue(dw.pool, max_stages=2)
    try:
        with pytest.raises(cp.CrossPoolError) as e:
            qu.push([1])                                  # MLA request
        assert e.value.status == cp.CP_ERR_UNSUPPORTED
        with pytest.raises(cp.CrossPoolError) as e:
            qu.push([0], dep_stage=0)                     # depends on a stage that does not exist yet
        assert e.value.status == cp.CP_ERR_INVALID_ARG
        assert qu.push([0]) == 0
        with pytest.raises(cp.CrossPoolError) as e:
            qu.push([0, 2], dep_stage=0)                  # other batch shape than its predecessor
        assert e.value.status == cp.CP_ERR_INVALID_ARG
        assert qu.push([2], dep_stage=0, alpha=0.5) == 1
        with pytest.raises(cp.CrossPoolError) as e:
            qu.push([0])                                  # ring full
        assert e.value.status == cp.CP_ERR_INVALID_ARG
        qu.close_queue()
    finally:
        qu.free()
        dw.close()
