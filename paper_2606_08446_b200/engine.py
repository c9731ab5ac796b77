"""Buffer owner + call sequencer for one batch: summarize -> select -> sparse decode (or dense decode).

This is plumbing only: it allocates device buffers with torch and calls the C ABI through ``binding``;
every step of the path runs in the CUDA kernels.  Importing it without the built library fails loudly.
"""
from __future__ import annotations

from typing import Optional

import torch

from . import binding as B
from .workloads import PAGE, Workload, full_page_updates


class SparrowEngine:
    def __init__(self, wl: Workload, schedule: Optional[dict] = None, want_scores: bool = False, landmark: str = "minmax",
                 kv_layout="hnd", deterministic=False):
        assert wl.q.is_cuda, "the engine needs the workload on a CUDA device (no CPU fallback)"
        self.wl = wl
        dev = wl.q.device
        self.landmark = landmark      # "minmax" (north_star's default, 512 B per page and head) or "mean" (the cost model's single vector, 256 B)
        # kv_layout: how wl.k_cache / wl.v_cache are laid out -- "hnd" (packed, the default), "nhd" or explicit element strides
        self.shape = B.make_shape(wl.n_seq, wl.Hq, wl.Hkv, wl.max_pages, wl.n_phys, page_size=wl.page_size, landmark=landmark,
                                  kv_layout=kv_layout, deterministic=deterministic)
        self.set_schedule(schedule or wl.schedule)
        self.summaries = torch.zeros((wl.n_phys, wl.Hkv, 2, 128) if landmark == "minmax" else (wl.n_phys, wl.Hkv, 128),
                                     dtype=torch.bfloat16, device=dev)
        self.sel_count = torch.zeros((wl.n_seq,), dtype=torch.int32, device=dev)
        self.out = torch.zeros((wl.n_seq, wl.Hq, 128), dtype=torch.bfloat16, device=dev)
        self.lse = torch.zeros((wl.n_seq, wl.Hq), dtype=torch.float32, device=dev)
        self.out_dense = torch.zeros_like(self.out)
        self.lse_dense = torch.zeros_like(self.lse)
        self.select_ws = torch.zeros((B.sparrow_select_workspace_bytes(self.shape),), dtype=torch.uint8, device=dev)
        self.scores = (torch.full((wl.n_seq, wl.Hkv, wl.max_pages), float("nan"), dtype=torch.float32, device=dev)
                       if want_scores else None)
        self.dense_ws = torch.zeros((B.sparrow_decode_workspace_bytes(self.shape, 0),), dtype=torch.uint8, device=dev)

    def set_schedule(self, spec: dict):
        dev = self.wl.q.device
        self.sched_spec = dict(spec)
        self.sched = B.make_schedule(spec, page_size=self.wl.page_size)
        max_len = int(self.wl.seq_lens.max().item())
        self._len_now = max_len          # host-side bound on the longest cached length (appends add to it)
        self._len_sized = max_len        # the length max_sel is sized for
        self.max_sel = max(1, B.sparrow_max_sel_pages(self.sched, max_len))
        self.sel_pages = torch.full((self.wl.n_seq, self.wl.Hkv, self.max_sel), -1, dtype=torch.int32, device=dev)
        self.sparse_ws = torch.zeros((B.sparrow_decode_workspace_bytes(self.shape, self.max_sel),), dtype=torch.uint8, device=dev)

    # ---- a1
    def summarize(self, page_ids: Optional[torch.Tensor], n_valid: Optional[torch.Tensor], n_update: Optional[int] = None, stream=None):
        n = int(page_ids.numel()) if page_ids is not None else int(n_update)
        return B.sparrow_summarize(self.wl.k_cache, self.summaries, page_ids, n_valid, n, self.shape, stream)

    def summarize_all(self, stream=None):
        """Post-prefill bulk call over every page the batch owns (partial last pages use n_valid)."""
        if getattr(self, "_ids", None) is None:          # built once on the host; later calls only launch the kernel
            ids, nv = full_page_updates(self.wl)
            dev = self.wl.q.device
            self._ids, self._nv = ids.to(dev), nv.to(dev)
        return self.summarize(self._ids, self._nv, stream=stream)

    # ---- a2-a5
    def select(self, q=None, stream=None):
        wl = self.wl
        return B.sparrow_select(wl.q if q is None else q, self.summaries, wl.page_table, wl.seq_lens, self.sched,
                                self.sel_pages, self.max_sel, self.sel_count, self.scores, self.select_ws, self.shape, stream)

    # ---- a6-a7
    def sparse_decode(self, q=None, stream=None, out=None, lse=None):
        wl = self.wl
        return B.sparrow_sparse_decode(wl.q if q is None else q, wl.k_cache, wl.v_cache, wl.page_table, wl.seq_lens,
                                       self.sel_pages, self.max_sel, self.sel_count, self.out if out is None else out,
                                       self.lse if lse is None else lse, wl.sm_scale, self.sparse_ws, self.shape, stream)

    # ---- a8
    def dense_decode(self, q=None, stream=None, out=None, lse=None):
        wl = self.wl
        return B.sparrow_dense_decode(wl.q if q is None else q, wl.k_cache, wl.v_cache, wl.page_table, wl.seq_lens,
                                      self.out_dense if out is None else out, self.lse_dense if lse is None else lse,
                                      wl.sm_scale, self.dense_ws, self.shape, stream)

    # ---- 8(f)-1: the rollout loop
    def append(self, k_new, v_new, stream=None):
        """Cache side of a rollout step: write the token's K/V at position L, L += 1, summarize the page if it filled."""
        wl = self.wl
        # sparrow_append leaves a sequence untouched when its page table is full, and sparrow_select clamps to max_sel:
        # both are silent on the device, so the bounds are enforced here on the host (the lengths themselves live on
        # the device; _len_now is their host-side upper bound)
        assert self._len_now + 1 <= wl.max_pages * wl.page_size, "append: the page table has no room for another token"
        assert self._len_now + 1 <= self._len_sized, "append: call reserve(n_steps) first (max_sel is sized for the current lengths)"
        self._len_now += 1
        return B.sparrow_append(k_new, v_new, wl.k_cache, wl.v_cache, self.summaries, wl.page_table, wl.seq_lens, self.shape, stream)

    def note_appended(self, n_tokens: int):
        """Tell the engine that n_tokens more tokens per sequence were (or will be) appended outside its view, e.g. by
        replaying a captured rollout graph again: keeps the host-side length bound, and its checks, in step."""
        assert self._len_now + n_tokens <= self._len_sized, "note_appended: beyond what reserve() sized the buffers for"
        self._len_now += n_tokens

    def reserve(self, n_steps: int):
        """Size the selection buffers for lengths up to the current maximum + n_steps (B(L) grows with L)."""
        self._len_now = int(self.wl.seq_lens.max().item())
        max_len = self._len_now + n_steps
        assert max_len <= self.wl.max_pages * self.wl.page_size, "the page table has no room for that many appended tokens"
        self._len_sized = max_len
        dev = self.wl.q.device
        self.max_sel = max(1, B.sparrow_max_sel_pages(self.sched, max_len))
        self.sel_pages = torch.full((self.wl.n_seq, self.wl.Hkv, self.max_sel), -1, dtype=torch.int32, device=dev)
        self.sparse_ws = torch.zeros((B.sparrow_decode_workspace_bytes(self.shape, self.max_sel),), dtype=torch.uint8, device=dev)

    def rollout(self, q_steps, k_steps, v_steps, out_steps, lse_steps=None, dense=False, stream=None):
        """T decode steps back to back on one stream (capturable as ONE CUDA graph: the lengths live on the device
        and every launch is asynchronous): append -> select -> sparse decode per step, or append -> dense decode."""
        for t in range(q_steps.shape[0]):
            self.append(k_steps[t], v_steps[t], stream)
            lse = None if lse_steps is None else lse_steps[t]
            if dense:
                self.dense_decode(q_steps[t], stream, out=out_steps[t], lse=self.lse_dense if lse is None else lse)
            else:
                self.select(q_steps[t], stream)
                self.sparse_decode(q_steps[t], stream, out=out_steps[t], lse=lse)
        return out_steps

    def step(self, q=None, updates=None, stream=None):
        """One pass of the hot path: summarize the pages that just filled, then select and sparse decode."""
        if updates is not None and updates[0].numel() > 0:
            self.summarize(updates[0], updates[1], stream=stream)
        self.select(q, stream)
        self.sparse_decode(q, stream)
        return self.out
