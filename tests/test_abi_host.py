"""CPU-side tests of libcrosspool: the library loads, exports every symbol the header
declares, and the host logic (validation, page ownership against the budget, all-or-nothing
mapping, the tile planner) behaves as include/crosspool.h states.  No compute call needs
a GPU here; on a box without CUDA the compute entry points must fail loudly."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2606_24506_b200 as cp
from workloads import KIND_KV, KIND_MLA, ModelCfg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FAKE_ARENA = 0x7F0000000000        # never dereferenced by host-side calls (256-B aligned)


def make_pool(P=16, num_pages=64, models=None, max_requests=8, max_ppr=64, page_bytes=None):
    models = models or [ModelCfg(KIND_KV, 8, 2, 128, 128, 0.1)]
    page_bytes = page_bytes or max(m.page_bytes(P) for m in models)
    return cp.Pool(FAKE_ARENA, num_pages * page_bytes, P, page_bytes, num_pages, models,
                   max_requests, max_ppr)


def test_library_exports_every_declared_symbol():
    L = cp.load_library()
    hdr = open(os.path.join(ROOT, "include", "crosspool.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(cp_[a-z_]+)\s*\(", hdr))
    assert declared == set(cp.EXPORTED), declared ^ set(cp.EXPORTED)
    for name in declared:
        assert getattr(L, name) is not None
    assert cp.status_string(0) == "CP_OK" and cp.status_string(-2) == "CP_ERR_NO_PAGES"


def test_create_validation():
    m = ModelCfg(KIND_KV, 8, 2, 128, 128, 0.1)
    with pytest.raises(cp.CrossPoolError) as e:
        cp.Pool(0, 1 << 20, 16, m.page_bytes(16), 8, [m], 4, 16)
    assert e.value.status == cp.CP_ERR_INVALID_ARG
    with pytest.raises(cp.CrossPoolError) as e:      # arena too small
        cp.Pool(FAKE_ARENA, 100, 16, m.page_bytes(16), 8, [m], 4, 16)
    assert e.value.status == cp.CP_ERR_INVALID_ARG
    with pytest.raises(cp.CrossPoolError) as e:      # misaligned arena
        cp.Pool(FAKE_ARENA + 16, 1 << 20, 16, m.page_bytes(16), 8, [m], 4, 16)
    assert e.value.status == cp.CP_ERR_INVALID_ARG
    for bad in (ModelCfg(KIND_KV, 8, 3, 128, 128, 0.1),        # Hq % Hkv
                ModelCfg(KIND_KV, 8, 2, 100, 128, 0.1),        # d not multiple of 8
                ModelCfg(KIND_MLA, 8, 2, 576, 512, 0.1),       # MLA with Hkv != 1
                ModelCfg(KIND_MLA, 8, 1, 64, 128, 0.1),        # MLA d_v > d_k
                ModelCfg(KIND_KV, 8, 2, 640, 128, 0.1)):       # d_k too large
        with pytest.raises(cp.CrossPoolError) as e:
            cp.Pool(FAKE_ARENA, 1 << 30, 16, 1 << 16, 8, [bad], 4, 16)
        assert e.value.status == cp.CP_ERR_UNSUPPORTED
    with pytest.raises(cp.CrossPoolError) as e:      # page does not fit
        cp.Pool(FAKE_ARENA, 1 << 30, 16, 4096, 8, [m], 4, 16)
    assert e.value.status == cp.CP_ERR_UNSUPPORTED


def test_map_unmap_ownership_and_budget():
    p = make_pool(P=16, num_pages=16, max_ppr=16)
    assert p.stats() == (16, 0)
    p.map_pages(0, 0, [3, 4, 5, 6], 20)               # 2 logical pages x 2 kv heads
    assert p.stats() == (12, 4)
    model, ctx, ids = p.request_info(0)
    assert (model, ctx, list(ids)) == (0, 20, [3, 4, 5, 6])

    def expect(status, *a, **k):
        before = (p.stats(), p.request_info(0))
        with pytest.raises(cp.CrossPoolError) as e:
            p.map_pages(*a, **k)
        assert e.value.status == status
        after = (p.stats(), p.request_info(0))
        assert before[0] == after[0] and list(before[1][2]) == list(after[1][2])   # unchanged

    expect(cp.CP_ERR_PAGE_IN_USE, 1, 0, [7, 3], 5)            # 3 owned by request 0
    expect(cp.CP_ERR_PAGE_IN_USE, 1, 0, [7, 7], 5)            # repeated in the list
    expect(cp.CP_ERR_PAGE_RANGE, 1, 0, [7, 16], 5)
    expect(cp.CP_ERR_PAGE_RANGE, 1, 0, [-1, 7], 5)
    expect(cp.CP_ERR_UNSUPPORTED, 1, 0, [7], 5)               # not a multiple of Hkv
    expect(cp.CP_ERR_INVALID_ARG, 1, 0, [7, 8], 17)           # ctx beyond mapped capacity
    expect(cp.CP_ERR_INVALID_ARG, 1, 0, [7, 8], 0)            # empty context (A8)
    expect(cp.CP_ERR_INVALID_ARG, 0, 0, None, 19)             # context never decreases
    expect(cp.CP_ERR_INVALID_ARG, 9, 0, [7, 8], 5)            # request id out of range
    expect(cp.CP_ERR_INVALID_ARG, 1, 3, [7, 8], 5)            # model id out of range
    expect(cp.CP_ERR_NO_PAGES, 1, 0, None, 5, n_allocate=14)  # budget: only 12 free -> reject
    expect(cp.CP_ERR_INVALID_ARG, 0, 0, [7] * 14, 21)         # exceeds max_pages_per_request

    p.map_pages(0, 0, None, 32)                               # ctx only
    p.map_pages(0, 0, [9, 8], 33)                             # append a logical page
    assert list(p.request_info(0)[2]) == [3, 4, 5, 6, 9, 8]
    p.map_pages(1, 0, None, 16, n_allocate=2)                 # library-allocated
    got = list(p.request_info(1)[2])
    assert len(set(got)) == 2 and not set(got) & {3, 4, 5, 6, 8, 9}
    assert p.stats() == (8, 8)
    with pytest.raises(cp.CrossPoolError) as e:
        p.unmap_request(2)
    assert e.value.status == cp.CP_ERR_UNKNOWN_REQUEST
    p.unmap_request(0)
    assert p.stats() == (14, 2)
    with pytest.raises(cp.CrossPoolError) as e:
        p.request_info(0)
    assert e.value.status == cp.CP_ERR_UNKNOWN_REQUEST
    p.map_pages(2, 0, [3, 4], 1)                              # freed pages are reusable
    p.close()


def _coverage(tiles, n_groups_expected, pages_of, near_equal=True):
    """every (batch, kv head) group's logical pages covered exactly once, splits contiguous and numbered in token order"""
    by_group = {}
    for (b, c, s, ns, p0, p1) in tiles:
        assert p1 > p0
        by_group.setdefault((b, c), []).append((s, ns, p0, p1))
    assert len(by_group) == n_groups_expected
    for (b, c), lst in by_group.items():
        lst.sort()
        assert [x[0] for x in lst] == list(range(lst[0][1]))
        pos = 0
        for (_, _, p0, p1) in lst:
            assert p0 == pos
            pos = p1
        assert pos == pages_of[b]
        lens = [x[3] - x[2] for x in lst]
        if near_equal:
            assert max(lens) - min(lens) <= 1            # near-equal splits


def _plan_pool():
    models = [ModelCfg(KIND_KV, 64, 8, 128, 128, 0.1), ModelCfg(KIND_KV, 16, 1, 128, 128, 0.1)]
    P = 32
    p = make_pool(P=P, num_pages=40000, models=models, max_requests=16, max_ppr=4096)
    ctxs = [129, 4000, 65, 16000, 31, 2048, 9000]
    mids = [0, 1, 0, 1, 1, 0, 0]
    pages_of = {}
    for i, (c, m) in enumerate(zip(ctxs, mids)):
        n = -(-c // P) * models[m].n_kv_heads
        p.map_pages(i, m, None, c, n_allocate=n)
        pages_of[i] = -(-c // P)
    return p, models, mids, pages_of


def test_tile_plan_covers_every_page_once_and_balances():
    """The near-equal-splits planner of the warp-MMA K/V kernel (CP_OPT_KERNEL = 3), the MLA and the generic kernels."""
    p, models, mids, pages_of = _plan_pool()
    p.set_option(cp.CP_OPT_KERNEL, 3)
    ids = list(range(len(mids)))
    tiles, n_groups = p.decode_plan(ids)
    assert n_groups == sum(models[m].n_kv_heads for m in mids)
    _coverage(tiles, n_groups, pages_of)
    lens = [t[5] - t[4] for t in tiles]
    assert lens == sorted(lens, reverse=True)        # longest first
    total = sum(lens)
    # one wave on 148 CTAs: at most one tile per CTA when the groups allow it, tile length within
    # [L_bal, 2 L_bal] of the balanced length L_bal = ceil(total / 148)
    assert 148 // 2 <= len(tiles) <= 148
    assert max(lens) <= 2 * -(-total // 148)
    p.set_option(cp.CP_OPT_WAVES_X16, 32)            # two waves
    tiles_w2, _ = p.decode_plan(ids)
    _coverage(tiles_w2, n_groups, pages_of)
    assert 148 < len(tiles_w2) <= 148 * 2
    # plan options
    p.set_option(cp.CP_OPT_NUM_CTAS, 4)
    p.set_option(cp.CP_OPT_WAVES_X16, 16)
    tiles2, _ = p.decode_plan(ids)
    _coverage(tiles2, n_groups, pages_of)
    assert len(tiles2) <= 4 + n_groups
    # batch subsets and order
    tiles3, ng3 = p.decode_plan([3, 0])
    _coverage(tiles3, 1 + 8, {0: pages_of[3], 1: pages_of[0]})
    # context growth across a page boundary invalidates the cached plan
    p.map_pages(3, 1, None, 16001, n_allocate=1)
    tiles4, _ = p.decode_plan([3, 0])
    _coverage(tiles4, 9, {0: pages_of[3] + 1, 1: pages_of[0]})
    assert p.counters()["plan_builds"] >= 4
    with pytest.raises(cp.CrossPoolError) as e:
        p.decode_plan([0, 0])
    assert e.value.status == cp.CP_ERR_INVALID_ARG
    with pytest.raises(cp.CrossPoolError) as e:
        p.decode_plan([0, 12])
    assert e.value.status == cp.CP_ERR_UNKNOWN_REQUEST
    p.close()


def test_tile_plan_of_the_tcgen05_kv_kernel_equal_pieces_and_tail():
    """Default planner of the MQA/GQA path: the groups' 128-token slices laid end to end and cut
    into n_ctas equal pieces whatever the group boundaries; with CP_OPT_STATIC_PCT < 100 the rest of every group
    forms short tiles for the dynamic list.  Tiles come in device order: static slot j of CTA b at j * n_ctas + b
    (empty slots are not reported), then the dynamic tiles, longest first."""
    p, models, mids, pages_of = _plan_pool()
    ids = list(range(len(mids)))
    P, pps = 32, 4
    tiles, n_groups = p.decode_plan(ids)
    assert n_groups == sum(models[m].n_kv_heads for m in mids)
    _coverage(tiles, n_groups, pages_of, near_equal=False)
    slices = lambda t: -(-(t[5] - t[4]) // pps)
    total = sum(-(-pages_of[i] // pps) * models[m].n_kv_heads for i, m in enumerate(mids))
    # every tile but a group's last is a whole number of slices, and starts on a slice boundary of its group
    for t in tiles:
        assert t[4] % pps == 0
        if t[2] != t[3] - 1:
            assert (t[5] - t[4]) % pps == 0
    # 148 pieces of floor/ceil(total / 148) slices: a piece is a run of consecutive tiles in token order, so the
    # tiles, re-sorted by position, can be cut into 148 runs whose lengths differ by at most the snapping slack
    assert sum(slices(t) for t in tiles) == total
    assert len(tiles) >= 148 and len(tiles) <= 148 + n_groups
    assert max(slices(t) for t in tiles) <= -(-total // 148) + 1
    # a quarter of every group left to the dynamic list, in tiles of at most 2 slices
    p.set_option(cp.CP_OPT_STATIC_PCT, 75)
    p.set_option(cp.CP_OPT_TAIL_TILE_SLICES, 2)
    tiles_t, _ = p.decode_plan(ids)
    _coverage(tiles_t, n_groups, pages_of, near_equal=False)
    n_tail = 0
    for i, m in enumerate(mids):
        n_sl = -(-pages_of[i] // pps)
        rest = n_sl - n_sl * 75 // 100
        n_tail += models[m].n_kv_heads * (-(-rest // 2) if rest >= 1 else 0)
    tail = tiles_t[len(tiles_t) - n_tail:]
    assert all(slices(t) <= 2 for t in tail)
    assert [slices(t) for t in tail] == sorted((slices(t) for t in tail), reverse=True)
    # a tail tile is the END of its group: every static tile of the group lies before it
    first_tail = {}
    for t in tail:
        first_tail[(t[0], t[1])] = min(first_tail.get((t[0], t[1]), 1 << 30), t[4])
    for t in tiles_t[:len(tiles_t) - n_tail]:
        assert t[5] <= first_tail.get((t[0], t[1]), 1 << 30)
    # few CTAs: the pieces follow the option, every CTA's share is equal to within one slice
    p.set_option(cp.CP_OPT_STATIC_PCT, 100)
    p.set_option(cp.CP_OPT_NUM_CTAS, 4)
    tiles4, _ = p.decode_plan(ids)
    _coverage(tiles4, n_groups, pages_of, near_equal=False)
    assert len(tiles4) <= 4 + n_groups
    p.set_option(cp.CP_OPT_MIN_TILE_PAGES, 64)        # cuts closer than 16 slices to a group boundary snap to it
    tiles5, _ = p.decode_plan(ids)
    _coverage(tiles5, n_groups, pages_of, near_equal=False)
    assert all(slices(t) >= 16 for t in tiles5 if t[3] > 1)        # no sliver next to a group boundary
    p.close()


def test_workspace_bytes_formula():
    m = ModelCfg(KIND_KV, 32, 1, 128, 128, 0.1)
    p = make_pool(P=64, num_pages=5000, models=[m], max_requests=2, max_ppr=4096)
    p.map_pages(0, 0, None, 4096 * 64, n_allocate=4096)
    tiles, ng = p.decode_plan([0])
    ns = tiles[0][3]
    assert ng == 1 and ns == len(tiles) and ns == 148           # one equal piece per CTA (2048 slices / 148)
    # per group: O[g][ns][d_v] + (m, l)[g][ns] floats (head-major partial layout)
    assert p.decode_workspace_bytes([0]) == ns * 32 * (128 + 2) * 4
    p.map_pages(1, 0, None, 64, n_allocate=1)       # single-tile request adds no workspace
    assert p.decode_workspace_bytes([1]) == 0
    p.close()


def test_compute_calls_fail_loudly_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present: covered by the gpu tests")
    p = make_pool()
    p.map_pages(0, 0, [0, 1], 10)
    buf = np.zeros(1 << 16, dtype=np.uint8)
    with pytest.raises(cp.CrossPoolError) as e:
        p.decode_attention([0], FAKE_ARENA, FAKE_ARENA, FAKE_ARENA, FAKE_ARENA, 1 << 20)
    assert e.value.status == cp.CP_ERR_CUDA
    with pytest.raises(cp.CrossPoolError) as e:
        p.gather_kv(0, FAKE_ARENA, FAKE_ARENA)
    assert e.value.status == cp.CP_ERR_CUDA
    p.close()


def test_append_kv_host_validation_is_all_or_nothing():
    """cp_pool_append_kv argument / budget errors are detected before anything changes (no GPU
    needed: the device is only touched after validation)."""
    models = [ModelCfg(KIND_KV, 8, 2, 128, 128, 0.1)]
    p = make_pool(P=16, num_pages=6, models=models, max_requests=4, max_ppr=8)
    p.map_pages(0, 0, None, 16, n_allocate=2)         # one full logical page (2 kv heads)
    p.map_pages(1, 0, None, 5, n_allocate=2)          # room left in its page
    p.map_pages(2, 0, None, 16, n_allocate=2)         # full page as well: pool is now exhausted
    before = (p.stats(), [p.request_info(i)[:2] for i in range(3)])
    k = np.zeros(3 * 2 * 128, dtype=np.uint16)
    with pytest.raises(cp.CrossPoolError) as e:       # requests 0 and 2 each need 2 fresh pages: 0 free
        p.append_kv([0, 1, 2], k, k)
    assert e.value.status == cp.CP_ERR_NO_PAGES
    with pytest.raises(cp.CrossPoolError) as e:
        p.append_kv([1, 3], k, k)
    assert e.value.status == cp.CP_ERR_UNKNOWN_REQUEST
    with pytest.raises(cp.CrossPoolError) as e:
        p.append_kv([1], None, k)
    assert e.value.status == cp.CP_ERR_INVALID_ARG
    with pytest.raises(cp.CrossPoolError) as e:       # KV-kind request without value rows
        p.append_kv([1], k, None)
    assert e.value.status == cp.CP_ERR_INVALID_ARG
    with pytest.raises(cp.CrossPoolError) as e:
        p.append_kv([1, 1], k, k)
    assert e.value.status == cp.CP_ERR_INVALID_ARG
    assert before == (p.stats(), [p.request_info(i)[:2] for i in range(3)])
    p.close()


def test_vmm_pool_fails_loudly_without_a_device():
    """cp_pool_create_vmm needs the driver (it reserves device virtual memory): argument errors are
    reported first, then CP_ERR_CUDA on a host without a GPU -- never a host-memory stand-in."""
    import torch
    m = ModelCfg(KIND_KV, 8, 1, 128, 128, 0.1)
    with pytest.raises(cp.CrossPoolError) as e:
        cp.Pool.create_vmm(0, 16, 8192, [m], 4, 64)
    assert e.value.status == cp.CP_ERR_INVALID_ARG
    with pytest.raises(cp.CrossPoolError) as e:
        cp.Pool.create_vmm(1 << 22, 16, 4096, [m], 4, 64)          # page too small for the model
    assert e.value.status == cp.CP_ERR_UNSUPPORTED
    if torch.cuda.is_available():
        pytest.skip("CUDA present: the VMM arena itself is covered by tests/test_gpu_vmm.py")
    with pytest.raises(cp.CrossPoolError) as e:
        cp.Pool.create_vmm(1 << 22, 16, 8192, [m], 4, 64)
    assert e.value.status == cp.CP_ERR_CUDA
    p = make_pool()
    with pytest.raises(cp.CrossPoolError) as e:
        p.vmm_info()
    assert e.value.status == cp.CP_ERR_INVALID_ARG
    p.close()


def test_planner_host_validation():
    """cp_planner_* argument checks happen before any CUDA call."""
    wsb = cp.planner_workspace_bytes(1000)
    assert wsb >= 4 * 65536 + 8 * 32 and wsb % 8 == 0
    assert cp.planner_workspace_bytes(0) < wsb < cp.planner_workspace_bytes(100000)
    a = FAKE_ARENA
    for offs, kap in (([0, 5, 3], [1.0, 1.0]),          # offsets decrease
                      ([1, 5], [1.0]),                  # do not start at 0
                      ([0, 5], [-1.0]),                 # negative kappa
                      ([0, 5], [float("nan")])):
        with pytest.raises(cp.CrossPoolError) as e:
            cp.planner_pool_demand(offs, kap, a, a, a, a, 4, a, a, a, wsb)
        assert e.value.status == cp.CP_ERR_INVALID_ARG
    with pytest.raises(cp.CrossPoolError) as e:
        cp.planner_pool_demand(list(range(0, 5 * 66, 5)), [1.0] * 65, a, a, a, a, 4, a, a, a, wsb)   # > 64 models
    assert e.value.status == cp.CP_ERR_INVALID_ARG
    with pytest.raises(cp.CrossPoolError) as e:
        cp.planner_pool_demand([0, 5], [1.0], a, a, a, a, 4, a, a, a, cp.planner_workspace_bytes(0))   # sized for no trace
    assert e.value.status == cp.CP_ERR_WORKSPACE
    cp.planner_pool_demand([0, 5], [1.0], a, a, a, a, 0, None, None, a, wsb)        # nothing to do: OK, no CUDA
    for n, q in ((0, 0.5), (10, 0.0), (10, 1.5)):
        with pytest.raises(cp.CrossPoolError) as e:
            cp.planner_quantile(a, n, q, 4096.0, a, wsb)
        assert e.value.status == cp.CP_ERR_INVALID_ARG
