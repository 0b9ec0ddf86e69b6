"""GPU tests of the CUDA-VMM-backed arena: the same hot path on
an arena the library reserves and backs chunk by chunk, each request in its own contiguous virtual
slot, the decode kernels computing page ids by arithmetic instead of reading the software table.
Parity bars are those of test_gpu_parity.py; results must also equal the caller-owned-arena path
bit for bit (same kernels, same tiles, same data)."""
import numpy as np
import pytest

import oracle
import workloads as W
from workloads import KIND_KV, KIND_MLA, ModelCfg
from test_gpu_parity import SMALL, compare, device_workload, torch_cuda  # noqa: F401

pytestmark = pytest.mark.gpu


def decode_once(w, options, **kw):
    dw = device_workload(w, **kw)
    try:
        for k, v in options.items():
            dw.pool.set_option(k, v)
        dw.out.fill_(float("nan"))
        dw.lse.fill_(float("nan"))
        dw.decode()
        return dw.results()
    finally:
        dw.close()


@pytest.mark.parametrize("case", [0, 1, 3, 4, 6, 8])
@pytest.mark.parametrize("kernel", [0, 1, 2])
def test_vmm_attention_small(torch_cuda, case, kernel):
    import paper_2606_24506_b200 as cp
    models, rm, rc, P, shift = SMALL[case]
    scale = 0.1 if models[0].kind == KIND_MLA and models[0].head_dim_qk == 576 else 1.0
    w = W.small_workload(models, rm, rc, page_tokens=P, seed=300 + case, value_scale=scale,
                         value_shift=shift, keep_contiguous=False)
    opts = {cp.CP_OPT_KERNEL: kernel, cp.CP_OPT_MIN_TILE_PAGES: 1}
    base = decode_once(w, opts)
    ref = oracle.decode_workload(w)
    for table in (0, 1):
        got = decode_once(w, {**opts, cp.CP_OPT_VMM_TABLE: table}, vmm=True)
        compare(w, got, ref, "vmm small%d/k%d/table%d" % (case, kernel, table))
        for (o, l), (bo, bl) in zip(got, base):
            assert np.array_equal(o, bo) and np.array_equal(l, bl), "VMM arena result differs from the table path"


@pytest.mark.parametrize("k", [2, 3, 4])
def test_vmm_attention_full_config(torch_cuda, k):
    w = W.config(k)
    got = decode_once(w, {}, vmm=True)
    worst = compare(w, got, oracle.decode_workload(w), "vmm cfg%d" % k)
    print("vmm cfg%d: %s" % (k, worst))


def test_vmm_gather_bit_exact(torch_cuda):
    models, rm, rc, P, _ = SMALL[3]
    w = W.small_workload(models, rm, rc, page_tokens=P, seed=77, keep_contiguous=False)
    dw = device_workload(w, vmm=True)
    try:
        for i, r in enumerate(w.requests):
            m = models[r.model_id]
            gk, gv = dw.gather(i)
            rk, rv = oracle.gather(w.arena, P, w.page_bytes, w.num_pages, m.kind, m.n_kv_heads, m.head_dim_qk,
                                   m.head_dim_v, r.page_ids, r.context_len)
            assert gk.tobytes() == rk.tobytes() and gv.tobytes() == rv.tobytes()
            # the page list the library built is the request's slot, in order
            _, _, ids = dw.pool.request_info(r.request_id)
            sp = dw.pool.vmm_info()["slot_pages"]
            assert np.array_equal(ids, r.request_id * sp + np.arange(r.page_ids.size))
    finally:
        dw.close()


def test_vmm_first_compute_call_with_slot_zero_unmapped(torch_cuda):
    """The base of the reserved range has no backing until request slot 0 is mapped: the first compute call of a
    pool whose only request sits in the LAST slot must still find the arena's device (taken from the arena
    object, not from the pointer) and give the right attention."""
    import torch
    import paper_2606_24506_b200 as cp
    from paper_2606_24506_b200.harness import raw_device_tensor
    m = ModelCfg(KIND_KV, 32, 4, 128, 128, 128 ** -0.5)
    w = W.small_workload([m], [0], [3000], page_tokens=64, seed=9, keep_contiguous=False)
    r = w.requests[0]
    n_req = 5
    torch.zeros(1, device="cuda:0")
    pool = cp.Pool.create_vmm(w.num_pages * w.page_bytes + (8 << 20), 64, w.page_bytes, w.models, n_req, r.page_ids.size)
    try:
        rid = n_req - 1
        pool.map_pages(rid, 0, None, r.context_len, n_allocate=r.page_ids.size)
        info = pool.vmm_info()
        pages = w.arena.reshape(w.num_pages, w.page_bytes // 2)
        src = torch.from_numpy(np.ascontiguousarray(pages[r.page_ids]).view(np.int16)).to("cuda:0")
        dst = raw_device_tensor(info["arena_dev"] + rid * info["slot_pages"] * w.page_bytes, src.numel() * 2, torch.device("cuda:0")).view(torch.int16)
        dst.copy_(src.reshape(-1))
        q = torch.from_numpy(w.q_packed().view(np.int16)).to("cuda:0")
        out = torch.full((32 * 128,), float("nan"), dtype=torch.float32, device="cuda:0")
        lse = torch.full((32,), float("nan"), dtype=torch.float32, device="cuda:0")
        need = max(pool.decode_workspace_bytes([rid]), 256)
        ws = torch.full((need,), 0xFF, dtype=torch.uint8, device="cuda:0")
        pool.decode_attention([rid], q, out, lse, ws, need, int(torch.cuda.current_stream().cuda_stream))
        torch.cuda.synchronize()
        (ro, rl), = oracle.decode_workload(w)
        o = out.cpu().numpy().reshape(32, 128)
        assert np.abs(o - ro).max() <= 1e-2 and np.linalg.norm(o - ro) / np.linalg.norm(ro) <= 1e-2
        assert np.abs(lse.cpu().numpy() - rl).max() <= 1e-3
    finally:
        pool.close()


def test_vmm_append_crosses_a_chunk_boundary(torch_cuda):
    """A request that grows token by token maps its next physical chunk when a new page falls past
    the backed prefix of its slot; K/V written on both sides of the boundary read back bit-exact and
    attention on the grown context tracks the oracle."""
    import torch
    m = ModelCfg(KIND_KV, 8, 1, 128, 128, 128 ** -0.5)
    P = 16
    w = W.small_workload([m], [0], [4090], page_tokens=P, seed=5, keep_contiguous=False, extra_pages=8)
    dw = device_workload(w, vmm=True, page_list_slack=4)
    try:
        info = dw.pool.vmm_info()
        pages_per_chunk = info["chunk_bytes"] // w.page_bytes
        assert w.requests[0].page_ids.size <= pages_per_chunk < w.requests[0].page_ids.size + 3, \
            "the case assumes the request starts just under one chunk (chunk %d B)" % info["chunk_bytes"]
        assert info["chunks_mapped"] == 1
        r = w.requests[0]
        rng = np.random.default_rng(3)
        # host image of the request's contiguous slot, grown with the oracle
        host = np.full((r.page_ids.size + 4) * (w.page_bytes // 2), W.BF16_NAN, dtype=np.uint16)
        host[:r.page_ids.size * (w.page_bytes // 2)] = w.arena.reshape(w.num_pages, -1)[r.page_ids].reshape(-1)
        ids = np.arange(r.page_ids.size, dtype=np.int32)
        ctx = r.context_len
        for step in range(3 * P):
            k = W.f32_to_bf16(rng.standard_normal((1, 128)).astype(np.float32))
            v = W.f32_to_bf16(rng.standard_normal((1, 128)).astype(np.float32))
            dw.pool.append_kv(dw.ids, torch.from_numpy(k.view(np.int16)).to(dw.device),
                              torch.from_numpy(v.view(np.int16)).to(dw.device), dw.stream())
            if ctx // P >= ids.size:
                ids = np.append(ids, np.int32(ids.size))
            oracle.append(host, P, w.page_bytes, r.page_ids.size + 4, m.kind, 1, 128, 128, ids, ctx, k, v)
            ctx += 1
        assert dw.pool.vmm_info()["chunks_mapped"] == 2
        _, c, lib_ids = dw.pool.request_info(0)
        assert c == ctx and np.array_equal(lib_ids, ids)          # slot 0: page ids are 0, 1, 2, ...
        w.arena, w.num_pages = host, r.page_ids.size + 4
        r.page_ids, r.context_len = ids, ctx
        gk, gv = dw.gather(0)
        rk, rv = oracle.gather(host, P, w.page_bytes, w.num_pages, m.kind, 1, 128, 128, ids, ctx)
        assert gk.tobytes() == rk.tobytes() and gv.tobytes() == rv.tobytes()
        dw.decode()
        compare(w, dw.results(), oracle.decode_workload(w), "vmm append")
    finally:
        dw.close()


def test_vmm_budget_admission_and_chunk_reuse(torch_cuda):
    """The physical budget is the pool page budget ("if the pool page budget is
    exhausted, admission control queues or rejects new requests"): a request the remaining chunks
    cannot back is rejected with nothing changed; after another request finishes, its parked chunks
    back the newcomer without new physical allocations."""
    import paper_2606_24506_b200 as cp
    torch_cuda.zeros(1, device="cuda:0")
    m = ModelCfg(KIND_KV, 8, 1, 128, 128, 128 ** -0.5)
    page_bytes = 16 * 256 * 2
    p = cp.Pool.create_vmm(2 * (2 << 20), 16, page_bytes, [m], max_requests=4, max_pages_per_request=1024)
    try:
        info = p.vmm_info()
        per_chunk = info["chunk_bytes"] // page_bytes
        assert info["chunks_budget"] * info["chunk_bytes"] <= 2 * (2 << 20) and info["chunks_mapped"] == 0
        budget = info["chunks_budget"]
        n_a = (budget - 1) * per_chunk + 1                     # needs every chunk of the budget
        p.map_pages(0, 0, None, n_a * 16, n_allocate=n_a)
        assert p.vmm_info()["chunks_mapped"] == budget
        with pytest.raises(cp.CrossPoolError) as e:
            p.map_pages(1, 0, None, 16, n_allocate=1)
        assert e.value.status == cp.CP_ERR_NO_PAGES
        with pytest.raises(cp.CrossPoolError) as e:
            p.request_info(1)
        assert e.value.status == cp.CP_ERR_UNKNOWN_REQUEST
        with pytest.raises(cp.CrossPoolError) as e:           # explicit page ids have no meaning here
            p.map_pages(1, 0, [5], 16)
        assert e.value.status == cp.CP_ERR_INVALID_ARG
        assert p.stats() == (0, n_a)
        p.unmap_request(0)
        assert p.vmm_info()["chunks_mapped"] == 0
        p.map_pages(1, 0, None, 16, n_allocate=1)
        assert p.vmm_info()["chunks_mapped"] == 1
        free, used = p.stats()
        assert used == 1 and free == (budget - 1) * per_chunk
    finally:
        p.close()
