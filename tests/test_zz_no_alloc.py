"""cp_planner_pool_demand_noalloc: the planner's pool-demand launches with their scratch in a static device
array of the library (for callers that cannot call cudaMalloc) against the existing path,
cp_planner_pool_demand with a caller-owned workspace.  Float64 with a fixed operation order on both paths,
so -- as in test_gpu_planner.py -- the bar is BIT-EXACT.  Two calls in a row on different traces: the array
keeps the first call's contents, the second must not see them.

Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

import oracle
from workloads.planner_traces import planner_trace


def bits(a):
    return np.ascontiguousarray(a, dtype=np.float64).view(np.uint64)


def to_dev(torch, tr, t_obs):
    return [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to("cuda:0")
            for a in (tr.arrival, tr.o_p, tr.o_d, tr.t_res, t_obs)]


@pytest.mark.gpu
def test_noalloc_pool_demand_matches_the_workspace_path_twice_in_a_row():
    import torch
    import paper_2606_24506_b200 as cp
    assert torch.cuda.is_available(), "gpu tests need a CUDA device (no CPU fallback exists)"
    stream = int(torch.cuda.current_stream().cuda_stream)
    # two traces of different shape: 8 models / long horizon, then 3 models / short horizon (fewer 32-entry blocks
    # and fewer models than the array still holds from the first call)
    cases = []
    for seed, n_models, horizon in ((31, 8, 2000.0), (32, 3, 400.0)):
        tr = planner_trace(seed, n_models=n_models, horizon_s=horizon, n_obs=2000)
        t_obs = np.concatenate([tr.t_obs, [-5.0, 0.0], tr.arrival[:20], (tr.arrival + tr.t_res)[:20], [horizon + 1e4]])
        assert 0 < tr.n_requests <= cp.PLANNER_NOALLOC_MAX_TRACE
        d = to_dev(torch, tr, t_obs)
        # the existing path, on a workspace of its own
        wsb = cp.planner_workspace_bytes(tr.n_requests)
        ws = torch.empty(wsb, dtype=torch.uint8, device="cuda:0")
        ref = torch.full((t_obs.size,), float("nan"), dtype=torch.float64, device="cuda:0")
        cp.planner_pool_demand(tr.offsets, tr.kappa, d[0], d[1], d[2], d[3], t_obs.size, d[4], ref, ws, wsb, stream)
        out = torch.full((t_obs.size,), float("nan"), dtype=torch.float64, device="cuda:0")
        cases.append((tr, t_obs, d, ref, out))
    torch.cuda.synchronize()

    def run_both():
        for tr, t_obs, d, _, out in cases:                 # back to back on one stream: ordered, no overlap
            out.fill_(float("nan"))
            cp.planner_pool_demand_noalloc(tr.offsets, tr.kappa, d[0], d[1], d[2], d[3], t_obs.size, d[4], out, stream)
        torch.cuda.synchronize()

    run_both()                                             # first use on this device: symbol address, module load
    free_before = torch.cuda.mem_get_info()[0]
    run_both()
    assert torch.cuda.mem_get_info()[0] == free_before, "the no-alloc entry point changed the device's free memory"
    for tr, t_obs, _, ref, out in cases:
        got = out.cpu().numpy()
        assert np.array_equal(bits(got), bits(ref.cpu().numpy())), "differs from cp_planner_pool_demand"
        assert got.max() > 0 and got[tr.t_obs.size] == 0.0 and got[-1] == 0.0
    # and the first trace once more after the second one, against the oracle this time
    tr, t_obs, d, _, out = cases[0]
    out.fill_(float("nan"))
    cp.planner_pool_demand_noalloc(tr.offsets, tr.kappa, d[0], d[1], d[2], d[3], t_obs.size, d[4], out, stream)
    torch.cuda.synchronize()
    exp = oracle.pool_demand(tr.offsets, tr.kappa, tr.arrival, tr.o_p, tr.o_d, tr.t_res, t_obs)
    assert np.array_equal(bits(out.cpu().numpy()), bits(exp))


def test_noalloc_pool_demand_rejects_what_does_not_fit():
    """A trace longer than the static array's capacity is refused before any CUDA call (runs without a GPU)."""
    import paper_2606_24506_b200 as cp
    big = cp.PLANNER_NOALLOC_MAX_TRACE + 1
    with pytest.raises(cp.CrossPoolError) as e:
        cp.planner_pool_demand_noalloc([0, big], [1.0], None, None, None, None, 4, None, None)
    assert e.value.status == cp.CP_ERR_TOO_LARGE
    assert cp.status_string(cp.CP_ERR_TOO_LARGE) == "CP_ERR_TOO_LARGE"
    with pytest.raises(cp.CrossPoolError) as e:            # the usual argument checks still apply
        cp.planner_pool_demand_noalloc(list(range(0, 5 * 66, 5)), [1.0] * 65, None, None, None, None, 4, None, None)
    assert e.value.status == cp.CP_ERR_INVALID_ARG
