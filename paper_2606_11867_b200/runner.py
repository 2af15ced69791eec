"""Device-buffer owner for one RL step: allocates the plan outputs and the assign workspace with
PyTorch (device memory and streams only) and forwards to the C-ABI calls of ``binding``.

No arithmetic of the method lives here; it exists so that tests, ``bench.py`` and users do not
repeat the allocation boilerplate.
"""
from __future__ import annotations

from typing import Optional

import torch

from . import binding as fm


class StepPlan:
    """Plan (a1-a4) of one step, resident on the device.

    ids int32 [L,T,K], w fp32 [L,T,K], mb_off int32 [n_mb+1], slot_expert int32 [L,S] (or
    [n_mb,L,S] with ``shape.placement_mb_stride = L*S``): CUDA tensors owned by the caller.
    """

    def __init__(self, shape: fm.Shape, ids, w, mb_off, slot_expert, want_step_hist: bool = True):
        dev = ids.device
        s = shape
        self.shape, self.ids, self.w, self.mb_off, self.slot_expert = s, ids, w, mb_off, slot_expert
        i32 = dict(dtype=torch.int32, device=dev)
        self.hist = torch.empty((s.n_mb, s.L, s.E), **i32)
        self.step_hist = (torch.empty((s.L, s.E), dtype=torch.int64, device=dev)
                          if want_step_hist else None)
        self.quota = torch.empty((s.n_mb, s.L, s.S), **i32)
        self.rank_load = torch.empty((s.n_mb, s.L, s.P), **i32)
        self.slot_off = torch.empty((s.n_mb, s.L, s.S + 1), **i32)
        self.pair_slot = torch.empty((s.L, s.T, s.K), **i32)
        self.inv = torch.empty((s.L, s.T, s.K), **i32)
        self.workspace = torch.empty(fm.workspace_bytes(s) + 16, dtype=torch.uint8, device=dev)
        self.status = torch.zeros(1, **i32)

    def load_hist(self) -> None:
        fm.load_hist(self.shape, self.ids, self.mb_off, self.hist, self.step_hist, self.status)

    def assign(self, quota_in: Optional[torch.Tensor] = None) -> None:
        fm.assign(self.shape, self.ids, self.mb_off, self.hist, self.slot_expert, quota_in,
                  self.quota, self.rank_load, self.slot_off, self.pair_slot, self.inv,
                  self.workspace, self.status)

    def plan(self, quota_in: Optional[torch.Tensor] = None) -> None:
        self.load_hist()
        self.assign(quota_in)

    def dispatch(self, layer: int, mb_begin: int, mb_end: int, x, perm, buf) -> None:
        fm.dispatch(self.shape, layer, mb_begin, mb_end, self.mb_off, self.inv, x, perm, buf,
                    self.status)

    def combine(self, layer: int, mb_begin: int, mb_end: int, expert_out, y) -> None:
        fm.combine(self.shape, layer, mb_begin, mb_end, self.mb_off, self.inv, self.w, expert_out,
                   y, self.status)

    def combine_bwd(self, layer: int, mb_begin: int, mb_end: int, dy, expert_out, d_expert_out,
                    dw=None) -> None:
        fm.combine_bwd(self.shape, layer, mb_begin, mb_end, self.mb_off, self.inv, self.w, dy,
                       expert_out, d_expert_out, dw, self.status)

    def dispatch_bwd(self, layer: int, mb_begin: int, mb_end: int, d_buf, dx) -> None:
        fm.dispatch_bwd(self.shape, layer, mb_begin, mb_end, self.mb_off, self.inv, d_buf, dx,
                        self.status)

    def faults(self) -> int:
        """Device fault bits raised so far (synchronises)."""
        return int(self.status.item())
