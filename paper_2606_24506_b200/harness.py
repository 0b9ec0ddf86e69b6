"""Device-side harness: put a host workload image into HBM and drive the C ABI.

Used by tests/, bench.py and __graft_entry__.smoke().  torch supplies device memory and
the stream only; nothing here computes any part of the attention.
"""
from __future__ import annotations

import numpy as np
import torch

from . import Pool


class _RawDeviceBytes:
    """CUDA array interface over a raw device address (memory the library mapped, not torch)."""

    def __init__(self, ptr: int, nbytes: int):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (ptr, False),
                                         "version": 3, "strides": None}


def raw_device_tensor(ptr: int, nbytes: int, device) -> torch.Tensor:
    """uint8 tensor view of `nbytes` at device address `ptr` (no copy, no ownership)."""
    return torch.as_tensor(_RawDeviceBytes(ptr, nbytes), device=device)


class DeviceWorkload:
    """A `workloads.Workload` resident on the GPU behind a cp_pool."""

    def __init__(self, w, device: str = "cuda:0", map_requests: bool = True, page_list_slack: int = 0,
                 vmm: bool = False, vmm_budget_bytes: int = 0):
        self.w = w
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        max_ppr = max(r.page_ids.size for r in w.requests) + page_list_slack    # room for appended pages
        self.vmm = vmm
        if vmm:
            # the library owns the arena (cp_pool_create_vmm): every request gets its contiguous virtual
            # slot, and the request's pages of the host image are copied there in page-list order
            torch.zeros(1, device=self.device)                       # make sure the context exists
            budget = vmm_budget_bytes or (w.num_pages * w.page_bytes + (len(w.requests) + 1) * (4 << 20))
            self.arena = None
            self.pool = Pool.create_vmm(budget, w.page_tokens, w.page_bytes, w.models,
                                        max_requests=len(w.requests), max_pages_per_request=max_ppr)
            if map_requests:
                info = self.pool.vmm_info()
                pages = w.arena.reshape(w.num_pages, w.page_bytes // 2)
                for r in w.requests:
                    self.pool.map_pages(r.request_id, r.model_id, None, r.context_len, n_allocate=r.page_ids.size)
                    src = torch.from_numpy(np.ascontiguousarray(pages[r.page_ids]).view(np.int16)).to(self.device)
                    dst = raw_device_tensor(info["arena_dev"] + r.request_id * info["slot_pages"] * w.page_bytes,
                                            src.numel() * 2, self.device).view(torch.int16)
                    dst.copy_(src.reshape(-1))
                torch.cuda.synchronize(self.device)
        else:
            # arena: one contiguous device buffer (torch allocations are >= 256-B aligned)
            self.arena = torch.from_numpy(w.arena.view(np.int16)).to(self.device)
            self.pool = Pool(self.arena, self.arena.numel() * 2, w.page_tokens, w.page_bytes, w.num_pages,
                             w.models, max_requests=len(w.requests), max_pages_per_request=max_ppr)
            if map_requests:
                for r in w.requests:
                    self.pool.map_pages(r.request_id, r.model_id, r.page_ids, r.context_len)
        self.ids = np.array([r.request_id for r in w.requests], dtype=np.int32)
        self.q = torch.from_numpy(w.q_packed().view(np.int16)).to(self.device)
        rows = w.out_rows()
        out_floats = sum(w.models[r.model_id].n_q_heads * w.models[r.model_id].head_dim_v
                         for r in w.requests)
        self.out = torch.empty(out_floats, dtype=torch.float32, device=self.device)
        self.lse = torch.empty(rows, dtype=torch.float32, device=self.device)
        self.ws_bytes = 0
        self.ws = None

    def stream(self) -> int:
        return int(torch.cuda.current_stream(self.device).cuda_stream)

    def ensure_workspace(self, ids=None):
        ids = self.ids if ids is None else ids
        need = self.pool.decode_workspace_bytes(ids)
        if self.ws is None or need > self.ws_bytes:
            self.ws_bytes = max(need, 256)
            self.ws = torch.empty(self.ws_bytes, dtype=torch.uint8, device=self.device)
        return need

    def decode(self, ids=None, q=None, out=None, lse=None):
        """One decode step on the current torch stream (asynchronous)."""
        ids = self.ids if ids is None else ids
        self.ensure_workspace(ids)
        self.pool.decode_attention(ids, self.q if q is None else q, self.out if out is None else out,
                                   self.lse if lse is None else lse, self.ws, self.ws_bytes,
                                   self.stream())

    def results(self):
        """Split the packed O / LSE into per-request numpy arrays (after a sync)."""
        torch.cuda.synchronize(self.device)
        o = self.out.cpu().numpy()
        l = self.lse.cpu().numpy()
        res, oo, lo = [], 0, 0
        for r in self.w.requests:
            m = self.w.models[r.model_id]
            n = m.n_q_heads * m.head_dim_v
            res.append((o[oo:oo + n].reshape(m.n_q_heads, m.head_dim_v).copy(),
                        l[lo:lo + m.n_q_heads].copy()))
            oo += n
            lo += m.n_q_heads
        return res

    def gather(self, i: int):
        r = self.w.requests[i]
        m = self.w.models[r.model_id]
        k = torch.empty((r.context_len, m.n_kv_heads, m.head_dim_qk), dtype=torch.int16, device=self.device)
        v = torch.empty((r.context_len, m.n_kv_heads, m.head_dim_v), dtype=torch.int16, device=self.device)
        self.pool.gather_kv(r.request_id, k, v, self.stream())
        torch.cuda.synchronize(self.device)
        return k.cpu().numpy().view(np.uint16), v.cpu().numpy().view(np.uint16)

    def close(self):
        self.pool.close()
