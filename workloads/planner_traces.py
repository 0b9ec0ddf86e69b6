"""Seeded synthetic request traces for the KV-cache planner.

Input generation only: nothing here evaluates Eq. (1)-(2) or a quantile.  The paper sizes the pool
from "per-model prompt, output, and service-time samples, arrival rate lambda_M, page size,
per-token KV bytes kappa(M)" taken from production traces that are not public; these stand-ins are
Poisson arrivals per cold model with lognormal prompt / output lengths and a decode residence
time that depends on both (so that the three stay correlated, which is what the trace-driven
quantile is meant to keep, L112).  The Monte-Carlo draws -- the observation times -- are part of
the generated input, so the oracle and the CUDA path consume the same numbers.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class PlannerTrace:
    offsets: np.ndarray      # int64 [M + 1]: model M owns entries offsets[M] .. offsets[M+1]-1
    kappa: np.ndarray        # float64 [M]  per-token KV bytes kappa(M)
    lam: np.ndarray          # float64 [M]  arrival rate (requests / s) the trace was drawn with
    arrival: np.ndarray      # float64 [N]  A_i, ascending inside each model
    o_p: np.ndarray          # float64 [N]  prompt tokens (integers stored as doubles)
    o_d: np.ndarray          # float64 [N]  output tokens
    t_res: np.ndarray        # float64 [N]  decode residence time T_i (s), > 0
    t_obs: np.ndarray        # float64 [n_obs] observation times (the Monte-Carlo draws)
    horizon: float

    @property
    def n_models(self) -> int:
        return int(self.kappa.size)

    @property
    def n_requests(self) -> int:
        return int(self.arrival.size)


# per-token KV bytes of the colocated model mix (bf16): 2 * layers * Hkv * 128 * 2 for K/V models,
# layers * 576 * 2 for an MLA model
KAPPA_CHOICES = np.array([2 * 32 * 8 * 128 * 2, 2 * 40 * 4 * 128 * 2, 2 * 48 * 1 * 128 * 2,
                          2 * 64 * 8 * 128 * 2, 61 * 576 * 2], dtype=np.float64)


def planner_trace(seed: int, n_models: int = 8, horizon_s: float = 7200.0, n_obs: int = 100000,
                  rate_range=(0.05, 1.0), prompt_median: float = 1200.0, output_median: float = 250.0,
                  warm_fraction: float = 0.1) -> PlannerTrace:
    rng = np.random.default_rng(seed)
    offsets = [0]
    arr, ops, ods, trs = [], [], [], []
    lam = np.exp(rng.uniform(np.log(rate_range[0]), np.log(rate_range[1]), n_models))
    kappa = KAPPA_CHOICES[rng.integers(0, KAPPA_CHOICES.size, n_models)]
    for m in range(n_models):
        n_draw = int(lam[m] * horizon_s * 1.3 + 50)
        a = np.cumsum(rng.exponential(1.0 / lam[m], n_draw))
        a = a[a < horizon_s]
        n = a.size
        shared = rng.standard_normal(n)                       # long prompts tend to come with long answers
        o_p = np.maximum(1.0, np.round(prompt_median * np.exp(1.0 * (0.6 * shared + 0.8 * rng.standard_normal(n)))))
        o_d = np.maximum(1.0, np.round(output_median * np.exp(0.8 * (0.6 * shared + 0.8 * rng.standard_normal(n)))))
        tpot = 0.03 * (1.0 + o_p / 8000.0) * np.exp(0.25 * rng.standard_normal(n))   # s per output token
        arr.append(a); ops.append(o_p); ods.append(o_d); trs.append(o_d * tpot)
        offsets.append(offsets[-1] + n)
    t_obs = rng.uniform(warm_fraction * horizon_s, horizon_s, n_obs)
    return PlannerTrace(np.array(offsets, dtype=np.int64), kappa, lam, np.concatenate(arr), np.concatenate(ops),
                        np.concatenate(ods), np.concatenate(trs), t_obs, float(horizon_s))
