"""GPU parity of cp_decode_attention_qlen (several query tokens per request, causal over the context's
last q_len tokens; the q_len > 1 variant SURVEY §8(f) N4 names) against oracle.attention_qlen, under the
bars of test_gpu_parity.py."""
import numpy as np
import pytest

import oracle
import workloads as W
from workloads import KIND_KV, KIND_MLA, ModelCfg
from test_gpu_parity import compare, device_workload, torch_cuda  # noqa: F401

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(180)]

GQA = ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5)
MQA = ModelCfg(KIND_KV, 16, 1, 128, 128, 128 ** -0.5)
MHA = ModelCfg(KIND_KV, 8, 8, 128, 128, 128 ** -0.5)


def run_qlen(torch, w, q_len, options=None, seed=0, vmm=False):
    import paper_2606_24506_b200 as cp
    rng = np.random.default_rng(1000 + seed)
    qs = [W.f32_to_bf16(rng.standard_normal((q_len, w.models[r.model_id].n_q_heads, 128)).astype(np.float32))
          for r in w.requests]
    dw = device_workload(w, vmm=vmm)
    try:
        for k, v in (options or {}).items():
            dw.pool.set_option(k, v)
        dev = dw.device
        q = torch.from_numpy(np.concatenate([x.reshape(-1) for x in qs]).view(np.int16)).to(dev)
        rows = sum(x.shape[0] * x.shape[1] for x in qs)
        out = torch.full((rows * 128,), float("nan"), dtype=torch.float32, device=dev)
        lse = torch.full((rows,), float("nan"), dtype=torch.float32, device=dev)
        wsb = max(dw.pool.decode_workspace_bytes_qlen(dw.ids, q_len), 256)
        ws = torch.full((wsb,), 0xFF, dtype=torch.uint8, device=dev)     # NaN patterns: nothing may be read unwritten
        dw.pool.decode_attention_qlen(dw.ids, q_len, q, out, lse, ws, wsb, dw.stream())
        torch.cuda.synchronize()
        o, l = out.cpu().numpy(), lse.cpu().numpy()
        out.fill_(float("nan"))
        ws.fill_(0xFF)
        dw.pool.decode_attention_qlen(dw.ids, q_len, q, out, lse, ws, wsb, dw.stream())
        torch.cuda.synchronize()
        assert np.array_equal(o, out.cpu().numpy()) and np.array_equal(l, lse.cpu().numpy()), "relaunch differs"
    finally:
        dw.close()
    got, ref, ro = [], [], 0
    for r, x in zip(w.requests, qs):
        m = w.models[r.model_id]
        n = q_len * m.n_q_heads
        got.append((o[ro * 128:(ro + n) * 128].reshape(n, 128).copy(), l[ro:ro + n].copy()))
        ro += n
        eo, el = oracle.attention_qlen(w.arena, w.page_tokens, w.page_bytes, w.num_pages, m.kind, m.n_q_heads,
                                       m.n_kv_heads, 128, 128, m.softmax_scale, r.page_ids, r.context_len, x)
        ref.append((eo.reshape(n, 128), el.reshape(n)))
    return compare(w, got, ref, "q_len=%d" % q_len)


CASES = [
    # (models, req_models, contexts, P, q_len)
    ([GQA], [0, 0, 0], [700, 33, 4], 16, 4),             # a context that is nothing but its query tokens
    ([GQA], [0, 0], [65, 1000], 64, 16),                 # 128 rows; the mask reaches back across a page boundary
    ([MQA], [0, 0, 0], [17, 2500, 130], 16, 3),          # 48 rows: three M tiles of a padded four
    ([MQA], [0], [3000], 128, 8),                        # 128 rows, one long request, many splits
    ([MHA, GQA, MQA], [0, 1, 2, 0], [410, 90, 1234, 5], 32, 5),
    ([GQA], [0], [2050], 32, 2),
    # groups of at most 32 rows: the tcgen05 K/V kernel (query rows on the MMA N dimension, causal limit per row)
    ([MHA], [0, 0, 0], [131, 258, 1000], 16, 7),         # last slice shorter than q_len - 1: the mask spans two slices
    ([GQA], [0], [128 * 20 + 2], 32, 4),                 # a last tile of two tokens that the first two query tokens do not see
    ([MHA, GQA], [0, 1, 0], [5000, 4099, 32], 64, 4),    # 4-row and 32-row groups in one launch
    ([MHA], [0, 0], [32, 777], 16, 32),                  # 32 rows of one head; a context of query tokens only
    ([GQA], [0, 0], [3, 12345], 128, 3),
]


@pytest.mark.parametrize("case", range(len(CASES)))
@pytest.mark.parametrize("n_ctas", [0, 3])
@pytest.mark.parametrize("kernel", [0, 2, 3])
def test_qlen_matches_oracle(torch_cuda, case, n_ctas, kernel):
    """kernel 0: the default choice (tcgen05 K/V kernel for groups of <= 16 rows, else the warp-MMA kernel);
    kernel 2: the tcgen05 kernel up to 32 rows; kernel 3: the warp-MMA kernel for every case."""
    import paper_2606_24506_b200 as cp
    models, rm, rc, P, q_len = CASES[case]
    w = W.small_workload(models, rm, rc, page_tokens=P, seed=500 + case, keep_contiguous=False)
    opts = {cp.CP_OPT_MIN_TILE_PAGES: 1, cp.CP_OPT_KERNEL: kernel}
    if n_ctas:
        opts[cp.CP_OPT_NUM_CTAS] = n_ctas
    worst = run_qlen(torch_cuda, w, q_len, opts, seed=case)
    print("case %d ctas %d kernel %d: %s" % (case, n_ctas, kernel, worst))


@pytest.mark.parametrize("case", [6, 7, 8, 10])
def test_qlen_with_dynamic_tail_tiles(torch_cuda, case):
    """Short tail tiles popped from the work counter: the last one may hold nothing but tokens that the first
    query tokens do not see (a split with m = -inf, l = 0 for those rows)."""
    import paper_2606_24506_b200 as cp
    models, rm, rc, P, q_len = CASES[case]
    w = W.small_workload(models, rm, rc, page_tokens=P, seed=500 + case, keep_contiguous=False)
    opts = {cp.CP_OPT_MIN_TILE_PAGES: 1, cp.CP_OPT_STATIC_PCT: 50, cp.CP_OPT_TAIL_TILE_SLICES: 1, cp.CP_OPT_KERNEL: 2}
    worst = run_qlen(torch_cuda, w, q_len, opts, seed=case)
    print("case %d tail tiles: %s" % (case, worst))


def test_qlen_one_is_the_single_token_step(torch_cuda):
    torch = torch_cuda
    w = W.small_workload([GQA, MQA], [0, 1, 0], [333, 1500, 64], page_tokens=32, seed=9, keep_contiguous=False)
    dw = device_workload(w)
    try:
        dw.decode()
        base = dw.results()
        out = torch.full_like(dw.out, float("nan"))
        lse = torch.full_like(dw.lse, float("nan"))
        dw.ensure_workspace()
        dw.pool.decode_attention_qlen(dw.ids, 1, dw.q, out, lse, dw.ws, dw.ws_bytes, dw.stream())
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), dw.out.cpu().numpy())
        assert np.array_equal(lse.cpu().numpy(), dw.lse.cpu().numpy())
        # and a plain step after a q_len > 1 step plans again for one token
        dw.pool.decode_workspace_bytes_qlen(dw.ids, 4)
        dw.out.fill_(float("nan"))
        dw.decode()
        for (o, l), (bo, bl) in zip(dw.results(), base):
            assert np.array_equal(o, bo) and np.array_equal(l, bl)
    finally:
        dw.close()


def test_qlen_argument_errors(torch_cuda):
    import paper_2606_24506_b200 as cp
    mla = ModelCfg(KIND_MLA, 16, 1, 576, 512, 0.07)
    w = W.small_workload([GQA, MQA, mla], [0, 1, 2], [100, 3, 64], page_tokens=64, seed=3, keep_contiguous=False,
                         value_scale=0.1)
    dw = device_workload(w)
    try:
        buf = torch_cuda.zeros(1 << 20, dtype=torch_cuda.float32, device=dw.device)
        for ids, q_len, status in (([0], 0, cp.CP_ERR_INVALID_ARG), ([0], 129, cp.CP_ERR_INVALID_ARG),
                                   ([1], 4, cp.CP_ERR_INVALID_ARG),          # context of 3 tokens
                                   ([0], 17, cp.CP_ERR_UNSUPPORTED),         # 8 heads x 17 tokens > 128 rows
                                   ([2], 2, cp.CP_ERR_UNSUPPORTED),          # MLA
                                   ([0, 0], 2, cp.CP_ERR_INVALID_ARG)):
            with pytest.raises(cp.CrossPoolError) as e:
                dw.pool.decode_attention_qlen(ids, q_len, buf, buf, buf, buf, buf.numel() * 4, dw.stream())
            assert e.value.status == status, (ids, q_len)
        dw.pool.set_option(cp.CP_OPT_KERNEL, 1)
        with pytest.raises(cp.CrossPoolError) as e:
            dw.pool.decode_attention_qlen([0], 2, buf, buf, buf, buf, buf.numel() * 4, dw.stream())
        assert e.value.status == cp.CP_ERR_UNSUPPORTED
    finally:
        dw.close()


def test_qlen_on_a_vmm_arena(torch_cuda):
    import paper_2606_24506_b200 as cp
    models, rm, rc, P, q_len = CASES[4]
    w = W.small_workload(models, rm, rc, page_tokens=P, seed=504, keep_contiguous=False)
    worst = run_qlen(torch_cuda, w, q_len, {cp.CP_OPT_MIN_TILE_PAGES: 1}, seed=4, vmm=True)
    print(worst)


@pytest.mark.parametrize("cfg", [2, 4])
def test_qlen_full_size(torch_cuda, cfg):
    """Full size, default options (what bench.py's `qlen` leg times): BASELINE cfg2 / cfg4 with four query
    tokens per request."""
    worst = run_qlen(torch_cuda, W.config(cfg), 4, seed=77)
    print("cfg%d q_len 4: %s" % (cfg, worst))
