"""paper_2606_24506_b200 -- thin Python binding of libcrosspool (include/crosspool.h).

B200-native (sm_100a) paged decode attention on CrossPool's shared KV-cache pool.
This module only marshals arguments: every step of the hot path runs in the CUDA
kernels behind the C ABI.  PyTorch is used by callers for device memory and streams
only.  There is no CPU fallback: if the shared library is missing or no CUDA device is
usable the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcrosspool.so")

CP_OK = 0
CP_ERR_INVALID_ARG = -1
CP_ERR_NO_PAGES = -2
CP_ERR_PAGE_RANGE = -3
CP_ERR_PAGE_IN_USE = -4
CP_ERR_UNKNOWN_REQUEST = -5
CP_ERR_UNSUPPORTED = -6
CP_ERR_WORKSPACE = -7
CP_ERR_CUDA = -8
CP_ERR_TOO_LARGE = -9
PLANNER_NOALLOC_MAX_TRACE = 1 << 20          # CP_PLANNER_NOALLOC_MAX_TRACE

CP_KIND_KV = 0
CP_KIND_MLA = 1

CP_OPT_KERNEL = 0
CP_OPT_NUM_CTAS = 1
CP_OPT_WAVES_X16 = 2
CP_OPT_MIN_TILE_PAGES = 3
CP_OPT_VMM_TABLE = 4
CP_OPT_HOST_ZERO_COPY = 5
CP_OPT_TIMELINE = 6
CP_OPT_STATIC_PCT = 7
CP_OPT_TAIL_TILE_SLICES = 8
TIMELINE_SLOTS = 16


class cp_model_cfg(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int32), ("n_q_heads", ctypes.c_int32),
                ("n_kv_heads", ctypes.c_int32), ("head_dim_qk", ctypes.c_int32),
                ("head_dim_v", ctypes.c_int32), ("softmax_scale", ctypes.c_float)]


class cp_tile_info(ctypes.Structure):
    _fields_ = [("batch_index", ctypes.c_int32), ("kv_head", ctypes.c_int32),
                ("split", ctypes.c_int32), ("n_splits", ctypes.c_int32),
                ("page_begin", ctypes.c_int32), ("page_end", ctypes.c_int32)]


class CrossPoolError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__("%s failed: %s (%d)" % (where, status_string(status), status))


_lib = None


def load_library():
    """dlopen libcrosspool.so (built in-tree by paper_2606_24506_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libcrosspool.so not built: run `python -m paper_2606_24506_b200.build` "
                          "(or __graft_entry__.build()); there is no fallback path")
    L = ctypes.CDLL(LIB_PATH)
    vp, i32, u32, u64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_uint32, ctypes.c_uint64
    i32p = ctypes.POINTER(ctypes.c_int32)
    u32p = ctypes.POINTER(ctypes.c_uint32)
    u64p = ctypes.POINTER(ctypes.c_uint64)
    sig = {
        "cp_pool_create": (i32, [vp, u64, u32, u32, u32, ctypes.POINTER(cp_model_cfg), i32, i32, i32,
                                 ctypes.POINTER(vp)]),
        "cp_pool_create_vmm": (i32, [u64, u32, u32, ctypes.POINTER(cp_model_cfg), i32, i32, i32,
                                     ctypes.POINTER(vp)]),
        "cp_pool_vmm_info": (i32, [vp, ctypes.POINTER(vp), u64p, u64p, u32p, u32p, u32p]),
        "cp_pool_free": (i32, [vp]),
        "cp_pool_map_pages": (i32, [vp, i32, i32, i32p, i32, i32]),
        "cp_pool_unmap_request": (i32, [vp, i32]),
        "cp_pool_request_info": (i32, [vp, i32, i32p, i32p, i32p, i32p, i32]),
        "cp_pool_stats": (i32, [vp, u32p, u32p]),
        "cp_pool_set_option": (i32, [vp, i32, ctypes.c_int64]),
        "cp_pool_gather_kv": (i32, [vp, i32, vp, vp, vp]),
        "cp_pool_append_kv": (i32, [vp, i32p, i32, vp, vp, vp]),
        "cp_decode_workspace_bytes": (i32, [vp, i32p, i32, u64p]),
        "cp_decode_attention": (i32, [vp, i32p, i32, vp, vp, vp, vp, u64, vp]),
        "cp_decode_workspace_bytes_host": (i32, [vp, i32p, i32, u64p]),
        "cp_decode_attention_host": (i32, [vp, i32p, i32, vp, vp, vp, vp, u64, vp]),
        "cp_decode_workspace_bytes_qlen": (i32, [vp, i32p, i32, i32, u64p]),
        "cp_decode_attention_qlen": (i32, [vp, i32p, i32, i32, vp, vp, vp, vp, u64, vp]),
        "cp_decode_stages_workspace_bytes": (i32, [vp, i32, i32p, i32p, i32p, u64p]),
        "cp_decode_attention_stages": (i32, [vp, i32, i32p, i32p, i32p, ctypes.c_float, vp, vp, vp, vp, u64, vp]),
        "cp_decode_attention_stages_gated": (i32, [vp, i32, i32p, i32p, i32p, ctypes.c_float, vp, vp, vp, vp, u64, vp,
                                                   vp, u32]),
        "cp_decode_stages_gate_status": (i32, [vp, vp, i32p]),
        "cp_decode_plan": (i32, [vp, i32p, i32, ctypes.POINTER(cp_tile_info), i32, i32p, i32p]),
        "cp_pool_counters": (i32, [vp, u64p, u64p, u64p]),
        "cp_pool_read_timeline": (i32, [vp, u64p, i32, i32p]),
        "cp_status_string": (ctypes.c_char_p, [i32]),
        "cp_decode_step_workspace_bytes": (i32, [vp, i32p, i32, u64p]),
        "cp_decode_step": (i32, [vp, i32p, i32, vp, vp, vp, vp, vp, vp, u64, vp]),
        "cp_queue_create": (i32, [vp, i32, ctypes.POINTER(vp)]),
        "cp_queue_launch": (i32, [vp, vp, vp, vp, vp, u64, ctypes.c_uint32, vp]),
        "cp_queue_push": (i32, [vp, i32p, i32, i32, ctypes.c_float, i32p]),
        "cp_queue_close": (i32, [vp]),
        "cp_queue_status": (i32, [vp, vp, i32p, i32p, i32p]),
        "cp_queue_free": (i32, [vp]),
        "cp_probe_globaltimer": (i32, [vp, vp]),
        "cp_probe_read_stream": (i32, [vp, u64, i32, vp, vp]),
        "cp_planner_workspace_bytes": (u64, [ctypes.c_int64]),
        "cp_planner_pool_demand": (i32, [i32, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_double),
                                         vp, vp, vp, vp, ctypes.c_int64, vp, vp, vp, u64, vp]),
        "cp_planner_pool_demand_noalloc": (i32, [i32, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_double),
                                                 vp, vp, vp, vp, ctypes.c_int64, vp, vp, vp]),
        "cp_planner_quantile": (i32, [vp, ctypes.c_int64, ctypes.c_double, ctypes.c_double, vp, u64,
                                      ctypes.POINTER(ctypes.c_double), u64p, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    _lib = L
    return L


EXPORTED = ["cp_pool_create", "cp_pool_create_vmm", "cp_pool_vmm_info", "cp_pool_free", "cp_pool_map_pages", "cp_pool_unmap_request",
            "cp_pool_request_info", "cp_pool_stats", "cp_pool_set_option", "cp_pool_gather_kv",
            "cp_pool_append_kv",
            "cp_decode_workspace_bytes", "cp_decode_attention", "cp_decode_workspace_bytes_host",
            "cp_decode_attention_host", "cp_decode_workspace_bytes_qlen", "cp_decode_attention_qlen",
            "cp_decode_stages_workspace_bytes", "cp_decode_attention_stages", "cp_decode_attention_stages_gated",
            "cp_decode_stages_gate_status", "cp_decode_plan", "cp_pool_counters", "cp_pool_read_timeline", "cp_status_string",
            "cp_probe_globaltimer", "cp_probe_read_stream", "cp_queue_create", "cp_queue_launch", "cp_queue_push",
            "cp_queue_close", "cp_queue_status", "cp_queue_free", "cp_decode_step_workspace_bytes", "cp_decode_step",
            "cp_planner_workspace_bytes", "cp_planner_pool_demand", "cp_planner_quantile",
            "cp_planner_pool_demand_noalloc"]


def status_string(status: int) -> str:
    return load_library().cp_status_string(int(status)).decode()


def _check(status: int, where: str):
    if status != CP_OK:
        raise CrossPoolError(status, where)


def _ids(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _i32p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def _ptr(x) -> int:
    """Raw address of a torch tensor / numpy array / int."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if isinstance(x, np.ndarray):
        return int(x.ctypes.data)
    raise TypeError(type(x))


class Pool:
    """Owner of one cp_pool handle; method names follow the C entry points."""

    def __init__(self, arena_dev, arena_bytes: int, page_tokens: int, page_bytes: int, num_pages: int,
                 models: Sequence, max_requests: int, max_pages_per_request: int):
        L = load_library()
        arr = (cp_model_cfg * len(models))()
        for i, m in enumerate(models):
            arr[i] = cp_model_cfg(int(m.kind), int(m.n_q_heads), int(m.n_kv_heads), int(m.head_dim_qk),
                                  int(m.head_dim_v), float(m.softmax_scale))
        h = ctypes.c_void_p()
        _check(L.cp_pool_create(_ptr(arena_dev), arena_bytes, page_tokens, page_bytes, num_pages, arr,
                                len(models), max_requests, max_pages_per_request, ctypes.byref(h)),
               "cp_pool_create")
        self._h = h
        self._L = L
        self._keep = arena_dev        # keep the arena tensor alive

    @staticmethod
    def _models_array(models):
        arr = (cp_model_cfg * len(models))()
        for i, m in enumerate(models):
            arr[i] = cp_model_cfg(int(m.kind), int(m.n_q_heads), int(m.n_kv_heads), int(m.head_dim_qk),
                                  int(m.head_dim_v), float(m.softmax_scale))
        return arr

    @classmethod
    def create_vmm(cls, physical_budget_bytes: int, page_tokens: int, page_bytes: int, models: Sequence,
                   max_requests: int, max_pages_per_request: int) -> "Pool":
        """cp_pool_create_vmm: the library owns the arena (CUDA virtual memory management)."""
        L = load_library()
        h = ctypes.c_void_p()
        _check(L.cp_pool_create_vmm(physical_budget_bytes, page_tokens, page_bytes, cls._models_array(models),
                                    len(models), max_requests, max_pages_per_request, ctypes.byref(h)),
               "cp_pool_create_vmm")
        self = cls.__new__(cls)
        self._h, self._L, self._keep = h, L, None
        return self

    def vmm_info(self):
        base = ctypes.c_void_p()
        va, chunk = ctypes.c_uint64(), ctypes.c_uint64()
        sp, cm, cb = ctypes.c_uint32(), ctypes.c_uint32(), ctypes.c_uint32()
        _check(self._L.cp_pool_vmm_info(self._h, ctypes.byref(base), ctypes.byref(va), ctypes.byref(chunk),
                                        ctypes.byref(sp), ctypes.byref(cm), ctypes.byref(cb)), "cp_pool_vmm_info")
        return {"arena_dev": int(base.value or 0), "va_bytes": va.value, "chunk_bytes": chunk.value,
                "slot_pages": sp.value, "chunks_mapped": cm.value, "chunks_budget": cb.value}

    def close(self):
        if getattr(self, "_h", None):
            self._L.cp_pool_free(self._h)
            self._h = None

    __del__ = close

    # --- slow path
    def map_pages(self, request_id: int, model_id: int, page_ids: Optional[Sequence[int]],
                  context_len: int, n_allocate: int = 0):
        if page_ids is None:
            st = self._L.cp_pool_map_pages(self._h, request_id, model_id, None, n_allocate, context_len)
        else:
            a = _ids(page_ids)
            st = self._L.cp_pool_map_pages(self._h, request_id, model_id, _i32p(a), a.size, context_len)
        _check(st, "cp_pool_map_pages")

    def unmap_request(self, request_id: int):
        _check(self._L.cp_pool_unmap_request(self._h, request_id), "cp_pool_unmap_request")

    def request_info(self, request_id: int):
        m, c, n = ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int32()
        _check(self._L.cp_pool_request_info(self._h, request_id, ctypes.byref(m), ctypes.byref(c),
                                            ctypes.byref(n), None, 0), "cp_pool_request_info")
        ids = np.empty(n.value, dtype=np.int32)
        if n.value:
            _check(self._L.cp_pool_request_info(self._h, request_id, None, None, None, _i32p(ids), n.value),
                   "cp_pool_request_info")
        return m.value, c.value, ids

    def stats(self):
        f, u = ctypes.c_uint32(), ctypes.c_uint32()
        _check(self._L.cp_pool_stats(self._h, ctypes.byref(f), ctypes.byref(u)), "cp_pool_stats")
        return f.value, u.value

    def set_option(self, key: int, value: int):
        _check(self._L.cp_pool_set_option(self._h, key, value), "cp_pool_set_option")

    def counters(self):
        a, b, c = ctypes.c_uint64(), ctypes.c_uint64(), ctypes.c_uint64()
        _check(self._L.cp_pool_counters(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)),
               "cp_pool_counters")
        return {"kernel_launches": a.value, "plan_builds": b.value, "metadata_h2d_bytes": c.value}

    def read_timeline(self) -> np.ndarray:
        """Per-CTA globaltimer stamps (ns) of the pool's last decode launch: uint64 [n_ctas][16]."""
        n = ctypes.c_int32()
        _check(self._L.cp_pool_read_timeline(self._h, None, 0, ctypes.byref(n)), "cp_pool_read_timeline")
        out = np.zeros((max(n.value, 1), TIMELINE_SLOTS), dtype=np.uint64)
        _check(self._L.cp_pool_read_timeline(self._h, out.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64)), n.value,
                                             ctypes.byref(n)), "cp_pool_read_timeline")
        return out[:n.value]

    # --- several query tokens per request (causal over the context's last q_len tokens)
    def decode_workspace_bytes_qlen(self, request_ids, q_len: int) -> int:
        ids = _ids(request_ids)
        out = ctypes.c_uint64()
        _check(self._L.cp_decode_workspace_bytes_qlen(self._h, _i32p(ids), ids.size, q_len, ctypes.byref(out)),
               "cp_decode_workspace_bytes_qlen")
        return int(out.value)

    def decode_attention_qlen(self, request_ids, q_len: int, q_dev, out_dev, lse_dev, workspace_dev,
                              workspace_bytes: int, stream: int = 0):
        ids = _ids(request_ids)
        _check(self._L.cp_decode_attention_qlen(self._h, _i32p(ids), ids.size, q_len, _ptr(q_dev), _ptr(out_dev),
                                                _ptr(lse_dev), _ptr(workspace_dev), workspace_bytes, stream),
               "cp_decode_attention_qlen")

    # --- several attention steps in one persistent launch (layer-wise stages)
    @staticmethod
    def _stage_args(stages, deps):
        sizes = _ids([len(st) for st in stages])
        ids = _ids(np.concatenate([np.asarray(st, dtype=np.int32) for st in stages]))
        deps = _ids(deps)
        if deps.size != sizes.size:
            raise ValueError("one dependency entry per stage")
        return sizes, ids, deps

    def decode_stages_workspace_bytes(self, stages, deps) -> int:
        sizes, ids, deps = self._stage_args(stages, deps)
        out = ctypes.c_uint64()
        _check(self._L.cp_decode_stages_workspace_bytes(self._h, sizes.size, _i32p(sizes), _i32p(ids), _i32p(deps),
                                                        ctypes.byref(out)), "cp_decode_stages_workspace_bytes")
        return int(out.value)

    def decode_attention_stages(self, stages, deps, alpha: float, q_dev, out_dev, lse_dev, workspace_dev,
                                workspace_bytes: int, stream: int = 0):
        sizes, ids, deps = self._stage_args(stages, deps)
        _check(self._L.cp_decode_attention_stages(self._h, sizes.size, _i32p(sizes), _i32p(ids), _i32p(deps),
                                                  float(alpha), _ptr(q_dev), _ptr(out_dev), _ptr(lse_dev),
                                                  _ptr(workspace_dev), workspace_bytes, stream),
               "cp_decode_attention_stages")

    def decode_attention_stages_gated(self, stages, deps, alpha: float, q_dev, out_dev, lse_dev, workspace_dev,
                                      workspace_bytes: int, stream: int, published_dev, timeout_ms: int):
        sizes, ids, deps = self._stage_args(stages, deps)
        _check(self._L.cp_decode_attention_stages_gated(self._h, sizes.size, _i32p(sizes), _i32p(ids), _i32p(deps),
                                                        float(alpha), _ptr(q_dev), _ptr(out_dev), _ptr(lse_dev),
                                                        _ptr(workspace_dev), workspace_bytes, stream,
                                                        _ptr(published_dev), timeout_ms),
               "cp_decode_attention_stages_gated")

    def decode_stages_gate_status(self, stream: int = 0) -> int:
        out = ctypes.c_int32()
        _check(self._L.cp_decode_stages_gate_status(self._h, stream, ctypes.byref(out)), "cp_decode_stages_gate_status")
        return int(out.value)

    def decode_plan(self, request_ids):
        ids = _ids(request_ids)
        nt, ng = ctypes.c_int32(), ctypes.c_int32()
        _check(self._L.cp_decode_plan(self._h, _i32p(ids), ids.size, None, 0, ctypes.byref(nt),
                                      ctypes.byref(ng)), "cp_decode_plan")
        tiles = (cp_tile_info * max(1, nt.value))()
        _check(self._L.cp_decode_plan(self._h, _i32p(ids), ids.size, tiles, nt.value, ctypes.byref(nt),
                                      ctypes.byref(ng)), "cp_decode_plan")
        return [(t.batch_index, t.kv_head, t.split, t.n_splits, t.page_begin, t.page_end)
                for t in tiles[:nt.value]], ng.value

    # --- device path
    def gather_kv(self, request_id: int, k_out_dev, v_out_dev, stream: int = 0):
        _check(self._L.cp_pool_gather_kv(self._h, request_id, _ptr(k_out_dev), _ptr(v_out_dev), stream),
               "cp_pool_gather_kv")

    def append_kv(self, request_ids, k_new_dev, v_new_dev, stream: int = 0):
        ids = _ids(request_ids)
        _check(self._L.cp_pool_append_kv(self._h, _i32p(ids), ids.size, _ptr(k_new_dev), _ptr(v_new_dev), stream),
               "cp_pool_append_kv")

    def decode_step_workspace_bytes(self, request_ids) -> int:
        ids = _ids(request_ids)
        out = ctypes.c_uint64()
        _check(self._L.cp_decode_step_workspace_bytes(self._h, _i32p(ids), ids.size, ctypes.byref(out)),
               "cp_decode_step_workspace_bytes")
        return int(out.value)

    def decode_step(self, request_ids, k_new_dev, v_new_dev, q_dev, out_dev, lse_dev, workspace_dev,
                    workspace_bytes: int, stream: int = 0):
        """Append one token per request and attend over the grown contexts (one call, one launch where fused)."""
        ids = _ids(request_ids)
        _check(self._L.cp_decode_step(self._h, _i32p(ids), ids.size, _ptr(k_new_dev), _ptr(v_new_dev), _ptr(q_dev),
                                      _ptr(out_dev), _ptr(lse_dev), _ptr(workspace_dev), workspace_bytes, stream),
               "cp_decode_step")

    def decode_workspace_bytes(self, request_ids) -> int:
        ids = _ids(request_ids)
        b = ctypes.c_uint64()
        _check(self._L.cp_decode_workspace_bytes(self._h, _i32p(ids), ids.size, ctypes.byref(b)),
               "cp_decode_workspace_bytes")
        return b.value

    def decode_attention(self, request_ids, q_dev, out_dev, lse_dev, workspace_dev, workspace_bytes: int,
                         stream: int = 0):
        ids = _ids(request_ids)
        _check(self._L.cp_decode_attention(self._h, _i32p(ids), ids.size, _ptr(q_dev), _ptr(out_dev),
                                           _ptr(lse_dev), _ptr(workspace_dev), workspace_bytes, stream),
               "cp_decode_attention")

    def decode_workspace_bytes_host(self, request_ids) -> int:
        ids = _ids(request_ids)
        b = ctypes.c_uint64()
        _check(self._L.cp_decode_workspace_bytes_host(self._h, _i32p(ids), ids.size, ctypes.byref(b)),
               "cp_decode_workspace_bytes_host")
        return b.value

    def decode_attention_host(self, request_ids, q_host, out_host, lse_host, workspace_dev,
                              workspace_bytes: int, stream: int = 0):
        ids = _ids(request_ids)
        _check(self._L.cp_decode_attention_host(self._h, _i32p(ids), ids.size, _ptr(q_host), _ptr(out_host),
                                                _ptr(lse_host), _ptr(workspace_dev), workspace_bytes, stream),
               "cp_decode_attention_host")


# ---------------------------------------------------------------- KV-cache planner (Eq. (1)-(2))
class Queue:
    """Request queue of one persistent launch (cp_queue_*): stages are pushed while the kernel runs."""

    def __init__(self, pool: "Pool", max_stages: int):
        self._L = load_library()
        h = ctypes.c_void_p()
        _check(self._L.cp_queue_create(pool._h, max_stages, ctypes.byref(h)), "cp_queue_create")
        self._h = h
        self.pool = pool

    def launch(self, q_dev, out_dev, lse_dev, workspace_dev, workspace_bytes: int, timeout_ms: int = 2000, stream: int = 0):
        _check(self._L.cp_queue_launch(self._h, _ptr(q_dev), _ptr(out_dev), _ptr(lse_dev), _ptr(workspace_dev),
                                       workspace_bytes, timeout_ms, stream), "cp_queue_launch")

    def push(self, request_ids, dep_stage: int = -1, alpha: float = 0.0) -> int:
        ids = _ids(request_ids)
        out = ctypes.c_int32()
        _check(self._L.cp_queue_push(self._h, _i32p(ids), ids.size, dep_stage, alpha, ctypes.byref(out)), "cp_queue_push")
        return int(out.value)

    def close_queue(self):
        _check(self._L.cp_queue_close(self._h), "cp_queue_close")

    def status(self, stream: int = 0):
        a, b, c = ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int32()
        _check(self._L.cp_queue_status(self._h, stream, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)), "cp_queue_status")
        return {"stages_planned": a.value, "tiles_planned": b.value, "error": c.value}

    def free(self):
        if self._h:
            self._L.cp_queue_free(self._h)
            self._h = None


def probe_globaltimer(stamp_dev, stream: int = 0):
    """One-thread kernel on `stream` that stores %globaltimer (ns) to the 8-byte device location stamp_dev."""
    _check(load_library().cp_probe_globaltimer(_ptr(stamp_dev), stream), "cp_probe_globaltimer")


def probe_read_stream(src_dev, nbytes: int, n_ctas: int, sink_dev, stream: int = 0):
    """Read nbytes of device memory once (16-byte loads, nothing written): the read-only HBM ceiling."""
    _check(load_library().cp_probe_read_stream(_ptr(src_dev), nbytes, n_ctas, _ptr(sink_dev), stream), "cp_probe_read_stream")


def planner_workspace_bytes(n_trace_entries: int = 0) -> int:
    return int(load_library().cp_planner_workspace_bytes(int(n_trace_entries)))


def planner_pool_demand(trace_offsets, kappa, arrival_dev, prompt_tokens_dev, output_tokens_dev, residence_dev,
                        n_obs: int, t_obs_dev, k_pool_dev, workspace_dev, workspace_bytes: int, stream: int = 0):
    """cp_planner_pool_demand: K_pool(t) at the caller's observation times (device float64 arrays)."""
    offs = np.ascontiguousarray(trace_offsets, dtype=np.int64)
    kap = np.ascontiguousarray(kappa, dtype=np.float64)
    if offs.size != kap.size + 1:
        raise ValueError("trace_offsets must have n_models + 1 entries")
    _check(load_library().cp_planner_pool_demand(
        kap.size, offs.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)),
        kap.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), _ptr(arrival_dev), _ptr(prompt_tokens_dev),
        _ptr(output_tokens_dev), _ptr(residence_dev), n_obs, _ptr(t_obs_dev), _ptr(k_pool_dev),
        _ptr(workspace_dev), workspace_bytes, stream), "cp_planner_pool_demand")


def planner_pool_demand_noalloc(trace_offsets, kappa, arrival_dev, prompt_tokens_dev, output_tokens_dev, residence_dev,
                                n_obs: int, t_obs_dev, k_pool_dev, stream: int = 0):
    """cp_planner_pool_demand_noalloc: the same without a workspace (scratch in a static device array of the
    library; traces of up to PLANNER_NOALLOC_MAX_TRACE entries; calls that overlap on the GPU race on it)."""
    offs = np.ascontiguousarray(trace_offsets, dtype=np.int64)
    kap = np.ascontiguousarray(kappa, dtype=np.float64)
    if offs.size != kap.size + 1:
        raise ValueError("trace_offsets must have n_models + 1 entries")
    _check(load_library().cp_planner_pool_demand_noalloc(
        kap.size, offs.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)),
        kap.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), _ptr(arrival_dev), _ptr(prompt_tokens_dev),
        _ptr(output_tokens_dev), _ptr(residence_dev), n_obs, _ptr(t_obs_dev), _ptr(k_pool_dev), stream),
        "cp_planner_pool_demand_noalloc")


def planner_quantile(values_dev, n: int, q: float, page_bytes: float, workspace_dev, workspace_bytes: int,
                     stream: int = 0):
    """cp_planner_quantile -> (x_(ceil(q n)), pages)."""
    val, pages = ctypes.c_double(), ctypes.c_uint64()
    _check(load_library().cp_planner_quantile(_ptr(values_dev), n, q, page_bytes, _ptr(workspace_dev),
                                              workspace_bytes, ctypes.byref(val), ctypes.byref(pages), stream),
           "cp_planner_quantile")
    return float(val.value), int(pages.value)
