"""Pins of the KV-cache planner oracle (oracle/cp_oracle.c, planner section) against what the paper's
Eq. (1)-(2) and the mathematics fix.  CPU only.

P14  a request worked by hand, and the ends of the indicator's interval
P15  the exact time integral of K_pool: kappa * sum_i T_i (O_p,i + O_d,i / 2)
P16  Eq. (2) is a plain sum over models; kappa scales linearly
P17  the empirical quantile against a sort, and its special cases; page rounding
P18  Little's law on a long Poisson trace: E[K_M] = lambda kappa E[T (O_p + O_d / 2)]
"""
import numpy as np
import pytest

import oracle
from workloads.planner_traces import planner_trace


def demand_one(t, a, op, od, T, kappa=1.0):
    return oracle.pool_demand([0, 1], [kappa], [a], [op], [od], [T], np.atleast_1d(t))


def test_p14_hand_worked_request():
    # O_p = 100 prompt tokens, O_d = 50 output tokens over T = 10 s: 100 at admission, 125 half way,
    # just under 150 at the end, nothing before arrival and nothing from T on (Eq. (1): 0 <= u < T)
    assert oracle.active_tokens(0.0, 100, 50, 10) == 100.0
    assert oracle.active_tokens(5.0, 100, 50, 10) == 125.0
    assert oracle.active_tokens(2.0, 100, 50, 10) == 110.0
    assert oracle.active_tokens(10.0, 100, 50, 10) == 0.0
    assert oracle.active_tokens(np.nextafter(10.0, 0.0), 100, 50, 10) == pytest.approx(150.0, rel=1e-12)
    assert oracle.active_tokens(-1e-9, 100, 50, 10) == 0.0
    assert oracle.active_tokens(11.0, 100, 50, 10) == 0.0
    # the same through K_pool(t) = kappa * Q(t - A): arrival at A = 3, kappa = 4 bytes / token
    got = demand_one([2.9, 3.0, 8.0, 12.999, 13.0, 20.0], 3.0, 100, 50, 10, kappa=4.0)
    assert got[0] == 0.0 and got[1] == 400.0 and got[2] == 500.0 and got[4] == 0.0 and got[5] == 0.0
    assert got[3] == pytest.approx(4 * (100 + 50 * 0.9999), rel=1e-12)
    # a transposed operand (O_d + O_p u / T) or a dropped term would not give these
    assert oracle.active_tokens(5.0, 7, 1000, 10) == 507.0


def test_p15_time_integral_closed_form():
    """int K_pool(t) dt over the whole line = sum_M kappa_M sum_i T_i (O_p,i + O_d,i / 2): every
    request contributes the area of a trapezoid.  A midpoint rule on a fine grid must reproduce it up
    to the jumps at interval ends (<= one cell each)."""
    tr = planner_trace(11, n_models=3, horizon_s=400.0, n_obs=1, rate_range=(0.2, 0.6))
    exact = 0.0
    for m in range(tr.n_models):
        s = slice(tr.offsets[m], tr.offsets[m + 1])
        exact += tr.kappa[m] * np.sum(tr.t_res[s] * (tr.o_p[s] + tr.o_d[s] / 2.0))
    t_end = float((tr.arrival + tr.t_res).max()) + 1.0
    n = 400000
    dt = t_end / n
    grid = (np.arange(n) + 0.5) * dt
    k = oracle.pool_demand(tr.offsets, tr.kappa, tr.arrival, tr.o_p, tr.o_d, tr.t_res, grid)
    approx = float(np.sum(k) * dt)
    kmax = np.repeat(tr.kappa, np.diff(tr.offsets)) * (tr.o_p + tr.o_d)
    bound = float(np.sum(kmax) * dt)                 # each jump misplaces at most one cell of its height
    assert abs(approx - exact) <= bound
    assert bound < 2e-3 * exact                      # so the pin is tight: a dropped O_d / 2 term is 5-10 %
    assert (k >= 0).all()


def test_p16_sum_over_models_and_kappa():
    tr = planner_trace(12, n_models=3, horizon_s=600.0, n_obs=500)
    full = oracle.pool_demand(tr.offsets, tr.kappa, tr.arrival, tr.o_p, tr.o_d, tr.t_res, tr.t_obs)
    parts = []
    for m in range(3):
        s = slice(tr.offsets[m], tr.offsets[m + 1])
        parts.append(oracle.pool_demand([0, s.stop - s.start], tr.kappa[m:m + 1], tr.arrival[s], tr.o_p[s],
                                        tr.o_d[s], tr.t_res[s], tr.t_obs))
    assert np.array_equal(full, (parts[0] + parts[1]) + parts[2])          # Eq. (2), models in index order
    twice = oracle.pool_demand(tr.offsets, 2.0 * tr.kappa, tr.arrival, tr.o_p, tr.o_d, tr.t_res, tr.t_obs)
    assert np.array_equal(twice, 2.0 * full)                               # exact: a power of two
    # brute force in numpy on the same trace (pairwise summation: compare to rounding)
    rep_k = np.repeat(tr.kappa, np.diff(tr.offsets))
    u = tr.t_obs[:, None] - tr.arrival[None, :]
    q = np.where((u >= 0) & (u < tr.t_res[None, :]), tr.o_p[None, :] + tr.o_d[None, :] * u / tr.t_res[None, :], 0.0)
    np.testing.assert_allclose(full, (q * rep_k[None, :]).sum(axis=1), rtol=1e-12)
    # shifting every arrival and every observation time by the same amount changes nothing (to rounding)
    sh = oracle.pool_demand(tr.offsets, tr.kappa, tr.arrival + 64.0, tr.o_p, tr.o_d, tr.t_res, tr.t_obs + 64.0)
    np.testing.assert_allclose(sh, full, rtol=1e-9)


def test_p17_quantile_and_page_rounding():
    rng = np.random.default_rng(5)
    for n in (1, 2, 7, 100, 1001):
        x = rng.lognormal(3.0, 1.0, n)
        xs = np.sort(x)
        for q in (0.01, 0.5, 0.95, 0.99, 1.0):
            k = min(n, max(1, int(np.ceil(q * n))))
            assert oracle.quantile(x, q) == xs[k - 1]
            # at least a fraction q of the sample is <= the quantile, and it is the smallest such value
            assert np.mean(x <= oracle.quantile(x, q)) >= q - 1e-12
            if k > 1:
                assert np.mean(x <= xs[k - 2]) < q
    assert oracle.quantile([4.0] * 9, 0.95) == 4.0
    assert oracle.quantile([1, 2, 3, 4], 1.0) == 4.0 and oracle.quantile([1, 2, 3, 4], 0.5) == 2.0
    assert oracle.quantile([3, 1, 3, 3, 2], 0.6) == 3.0                     # ties
    qs = [oracle.quantile(np.arange(500.0), q) for q in (0.5, 0.9, 0.95, 0.99)]
    assert qs == sorted(qs) and qs == [249.0, 449.0, 474.0, 494.0]
    with pytest.raises(ValueError):
        oracle.quantile([1.0], 0.0)
    assert oracle.page_budget(0.0, 4096) == 0 and oracle.page_budget(1.0, 4096) == 1
    assert oracle.page_budget(4096.0, 4096) == 1 and oracle.page_budget(4097.0, 4096) == 2


def test_p18_littles_law_on_a_long_poisson_trace():
    """Campbell / Little: for Poisson arrivals of rate lambda the stationary mean of K_M is
    lambda * kappa * E[T (O_p + O_d / 2)].  Checked per model on a 40 000 s trace with the sample mean
    in place of the expectation (the trace's own realised rate), to a few per cent."""
    tr = planner_trace(13, n_models=2, horizon_s=40000.0, n_obs=6000, rate_range=(0.3, 0.5), warm_fraction=0.05)
    for m in range(2):
        s = slice(tr.offsets[m], tr.offsets[m + 1])
        n = s.stop - s.start
        k = oracle.pool_demand([0, n], tr.kappa[m:m + 1], tr.arrival[s], tr.o_p[s], tr.o_d[s], tr.t_res[s], tr.t_obs)
        rate = n / tr.horizon
        expect = rate * tr.kappa[m] * np.mean(tr.t_res[s] * (tr.o_p[s] + tr.o_d[s] / 2.0))
        assert abs(k.mean() - expect) < 0.06 * expect, (k.mean(), expect)
        assert abs(rate - tr.lam[m]) < 0.05 * tr.lam[m]
