"""Seeded random sweep of the single-step path: model shapes, page sizes, context mixes and scheduler
options drawn at random, every case compared with the oracle under the bars of test_gpu_parity.py.
The fixed cases elsewhere pin known edges; this one looks for the edges nobody listed."""
import numpy as np
import pytest

import workloads as W
from workloads import KIND_KV, KIND_MLA, ModelCfg
from test_gpu_parity import run_and_compare, torch_cuda  # noqa: F401

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(300)]


def draw_case(seed):
    import paper_2606_24506_b200 as cp
    rng = np.random.default_rng(9000 + seed)
    family = ["kv128", "kv128", "kv_generic", "mla", "mixed"][seed % 5]
    if family == "mla":
        P = int(rng.choice([32, 64, 128]))
        models = [ModelCfg(KIND_MLA, int(rng.choice([16, 64, 128])), 1, 576, 512, 192 ** -0.5)]
        scale = 0.1
    elif family == "kv_generic":
        P = int(rng.choice([8, 16, 32]))
        dk, dv = [(64, 64), (32, 16), (96, 64), (64, 128)][int(rng.integers(4))]
        hkv = int(rng.choice([1, 2, 3]))
        models = [ModelCfg(KIND_KV, hkv * int(rng.choice([1, 2, 5])), hkv, dk, dv, float(rng.uniform(0.05, 0.3)))]
        scale = 1.0
    else:
        P = int(rng.choice([16, 32, 64, 128]))
        models = []
        for _ in range(int(rng.integers(1, 4))):
            hkv = int(rng.choice([1, 2, 4, 8]))
            g = int(rng.choice([1, 2, 4, 5, 8, 12, 16, 32]))
            models.append(ModelCfg(KIND_KV, hkv * g, hkv, 128, 128, 128 ** -0.5))
        if family == "mixed":
            models.append(ModelCfg(KIND_KV, 6, 2, 64, 32, 0.2))
        scale = 1.0
    n_req = int(rng.integers(1, 7))
    rm = [int(rng.integers(len(models))) for _ in range(n_req)]
    rc = [int(np.exp(rng.uniform(0.0, np.log(6000.0)))) for _ in range(n_req)]
    rc = [max(1, c) for c in rc]
    if rng.random() < 0.5:
        rc[0] = int(rng.choice([1, P - 1, P, P + 1, 2 * P]))          # page-boundary contexts
    opts = {cp.CP_OPT_KERNEL: int(rng.choice([0, 0, 1, 2, 3])),
            cp.CP_OPT_STATIC_PCT: int(rng.choice([100, 100, 80, 50, 0])),
            cp.CP_OPT_TAIL_TILE_SLICES: int(rng.choice([1, 2, 5])),
            cp.CP_OPT_MIN_TILE_PAGES: int(rng.choice([1, 2, 4])),
            cp.CP_OPT_NUM_CTAS: int(rng.choice([0, 0, 3, 17, 100])),
            cp.CP_OPT_WAVES_X16: int(rng.choice([16, 8, 40]))}
    return family, models, rm, rc, P, scale, opts


@pytest.mark.parametrize("seed", range(60))
def test_random_case(torch_cuda, seed):
    family, models, rm, rc, P, scale, opts = draw_case(seed)
    w = W.small_workload(models, rm, rc, page_tokens=P, seed=7000 + seed, value_scale=scale,
                         value_shift=float(seed % 3), keep_contiguous=False)
    worst = run_and_compare(w, "sweep %d (%s)" % (seed, family), opts)
    print("seed %d %s P=%d ctx=%s opts=%s: %s" % (seed, family, P, rc, opts, worst))
