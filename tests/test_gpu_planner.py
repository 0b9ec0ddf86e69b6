"""GPU parity of the KV-cache planner (Eq. (1)-(2), L103-L114) against the
CPU oracle through the C ABI.  Float64 on both sides, every operation rounded separately in the
paper's order: the demand vector and the selected quantile must be BIT-EXACT, the page budget equal."""
import numpy as np
import pytest

import oracle
from workloads.planner_traces import planner_trace

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device (no CPU fallback exists)"
    return torch


def gpu_demand(torch, tr, t_obs=None):
    import paper_2606_24506_b200 as cp
    dev = "cuda:0"
    t_obs = tr.t_obs if t_obs is None else np.ascontiguousarray(t_obs, dtype=np.float64)
    d = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (tr.arrival, tr.o_p, tr.o_d, tr.t_res, t_obs)]
    out = torch.full((t_obs.size,), float("nan"), dtype=torch.float64, device=dev)
    wsb = cp.planner_workspace_bytes(tr.n_requests)
    ws = torch.empty(wsb, dtype=torch.uint8, device=dev)
    cp.planner_pool_demand(tr.offsets, tr.kappa, d[0], d[1], d[2], d[3], t_obs.size, d[4], out, ws, wsb,
                           int(torch.cuda.current_stream().cuda_stream))
    torch.cuda.synchronize()
    return out, ws, wsb


def bits(a):
    return np.ascontiguousarray(a, dtype=np.float64).view(np.uint64)


@pytest.mark.parametrize("seed,n_models,horizon", [(21, 1, 300.0), (22, 3, 900.0), (23, 8, 2000.0)])
def test_pool_demand_bit_exact(torch_cuda, seed, n_models, horizon):
    tr = planner_trace(seed, n_models=n_models, horizon_s=horizon, n_obs=3000)
    # observation times also before the first arrival, at exact arrival instants and at exact interval ends
    extra = np.concatenate([[-5.0, 0.0], tr.arrival[:50], (tr.arrival + tr.t_res)[:50], [horizon + 1e4]])
    t_obs = np.concatenate([tr.t_obs, extra])
    got, _, _ = gpu_demand(torch_cuda, tr, t_obs)
    ref = oracle.pool_demand(tr.offsets, tr.kappa, tr.arrival, tr.o_p, tr.o_d, tr.t_res, t_obs)
    assert np.array_equal(bits(got.cpu().numpy()), bits(ref))
    n0 = tr.t_obs.size                                   # t = -5 and t = 0 precede every arrival; the last is long after
    assert ref[n0] == 0.0 and ref[n0 + 1] == 0.0 and ref[-1] == 0.0 and ref.max() > 0


def test_pool_demand_edge_cases(torch_cuda):
    import paper_2606_24506_b200 as cp
    tr = planner_trace(24, n_models=3, horizon_s=500.0, n_obs=200)
    # a model without requests, a request with T = 0 (contributes nothing), simultaneous arrivals
    n1, n2, n3 = (int(x) for x in tr.offsets[1:])
    keep = np.r_[0:n1, n2:n3]                         # drop model 1's requests: it stays in the list, empty
    tr.arrival, tr.o_p, tr.o_d, tr.t_res = (a[keep].copy() for a in (tr.arrival, tr.o_p, tr.o_d, tr.t_res))
    tr.offsets = np.array([0, n1, n1, n1 + n3 - n2], dtype=np.int64)
    tr.t_res[3] = 0.0
    tr.arrival[5] = tr.arrival[4]
    got, ws, wsb = gpu_demand(torch_cuda, tr)
    ref = oracle.pool_demand(tr.offsets, tr.kappa, tr.arrival, tr.o_p, tr.o_d, tr.t_res, tr.t_obs)
    assert np.array_equal(bits(got.cpu().numpy()), bits(ref))
    # n_obs = 0 is a no-op; too small a workspace is rejected
    cp.planner_pool_demand(tr.offsets, tr.kappa, got, got, got, got, 0, None, None, ws, wsb)
    with pytest.raises(cp.CrossPoolError) as e:
        cp.planner_pool_demand(tr.offsets, tr.kappa, got, got, got, got, 1, got, got, ws, 1024)
    assert e.value.status == cp.CP_ERR_WORKSPACE


def test_quantile_bit_exact(torch_cuda):
    import paper_2606_24506_b200 as cp
    torch = torch_cuda
    rng = np.random.default_rng(31)
    wsb = cp.planner_workspace_bytes()
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda:0")
    cases = [rng.lognormal(20.0, 1.0, 1), rng.lognormal(20.0, 1.0, 2), rng.lognormal(20.0, 2.0, 1001),
             np.full(777, 3.5), np.floor(rng.uniform(0, 4, 5000)),             # constant / heavy ties
             np.concatenate([np.zeros(100), rng.uniform(0, 1e-300, 100)]),     # zeros and tiny values
             rng.lognormal(24.0, 0.7, 300000)]
    for x in cases:
        xd = torch.from_numpy(x).to("cuda:0")
        for q in (0.001, 0.5, 0.95, 0.99, 1.0):
            val, pages = cp.planner_quantile(xd, x.size, q, 16384.0, ws, wsb)
            ref = oracle.quantile(x, q)
            assert bits([val])[0] == bits([ref])[0], (x.size, q, val, ref)
            assert pages == oracle.page_budget(ref, 16384.0)
        assert np.array_equal(xd.cpu().numpy(), x)                             # input untouched
    with pytest.raises(cp.CrossPoolError) as e:
        cp.planner_quantile(xd, 0, 0.5, 1.0, ws, wsb)
    assert e.value.status == cp.CP_ERR_INVALID_ARG


def test_planner_full_size_budget(torch_cuda):
    """The planner run bench.py times: 8 cold models, two hours of trace, 100 000 observation times.
    The oracle evaluates every observation too (a few seconds): demand bit-exact, P95 / P99 and the page
    budgets equal, and the budget admits exactly what it should (pages * page_bytes >= K_q > (pages-1) * ...)."""
    import paper_2606_24506_b200 as cp
    tr = planner_trace(1)
    got, ws, wsb = gpu_demand(torch_cuda, tr)
    ref = oracle.pool_demand(tr.offsets, tr.kappa, tr.arrival, tr.o_p, tr.o_d, tr.t_res, tr.t_obs)
    assert np.array_equal(bits(got.cpu().numpy()), bits(ref))
    page_bytes = 64 * 256 * 2.0
    last = 0
    for q in (0.95, 0.99):
        val, pages = cp.planner_quantile(got, tr.t_obs.size, q, page_bytes, ws, wsb)
        assert val == oracle.quantile(ref, q) and pages == oracle.page_budget(val, page_bytes)
        assert pages * page_bytes >= val > (pages - 1) * page_bytes
        assert np.mean(ref <= val) >= q
        assert pages >= last
        last = pages
    print("P99 demand %.2f GiB -> %d pages" % (val / 2 ** 30, pages))
