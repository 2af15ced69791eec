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
        self._dp = None

    def data_path(self) -> fm.DataPath:
        """The data-path calls with this plan's arguments marshalled once (binding.DataPath)."""
        if self._dp is None:
            self._dp = fm.DataPath(self.shape, self.mb_off, self.inv, self.w, self.status)
        return self._dp

    def load_hist(self) -> None:
        fm.load_hist(self.shape, self.ids, self.mb_off, self.hist, self.step_hist, self.status)

    def assign(self, quota_in: Optional[torch.Tensor] = None) -> None:
        fm.assign(self.shape, self.ids, self.mb_off, self.hist, self.slot_expert, quota_in,
                  self.quota, self.rank_load, self.slot_off, self.pair_slot, self.inv,
                  self.workspace, self.status)

    def plan(self, quota_in: Optional[torch.Tensor] = None) -> None:
        """a1-a4 for a given placement: foremoe_plan (two passes over the ids, same results as
        load_hist() + assign())."""
        fm.plan(self.shape, self.ids, self.mb_off, self.slot_expert, quota_in, self.hist, self.step_hist,
                self.quota, self.rank_load, self.slot_off, self.pair_slot, self.inv, self.workspace,
                self.status)

    def dispatch(self, layer: int, mb_begin: int, mb_end: int, x, perm, buf) -> None:
        self.data_path().dispatch(layer, mb_begin, mb_end, x, perm, buf)

    def combine(self, layer: int, mb_begin: int, mb_end: int, expert_out, y) -> None:
        self.data_path().combine(layer, mb_begin, mb_end, expert_out, y)

    def combine_bwd(self, layer: int, mb_begin: int, mb_end: int, dy, expert_out, d_expert_out,
                    dw=None) -> None:
        self.data_path().combine_bwd(layer, mb_begin, mb_end, dy, expert_out, d_expert_out, dw)

    def dispatch_bwd(self, layer: int, mb_begin: int, mb_end: int, d_buf, dx) -> None:
        self.data_path().dispatch_bwd(layer, mb_begin, mb_end, d_buf, dx)

    def faults(self) -> int:
        """Device fault bits raised so far (synchronises)."""
        return int(self.status.item())


class LocalStepPlan(StepPlan):
    """Per-source, multi-machine plan: the StepPlan of the commodity
    instance (expert, source machine).  ``shape`` is the REAL shape, ``tok_src`` int32 [T] the source
    rank of every token, ``M`` the number of machines.  Every attribute of StepPlan then refers to
    the virtual instance (``hist`` [n_mb,L,E*M], ``quota`` [n_mb,L,S*M], ``pair_slot`` = slot*M +
    source machine); ``inv`` / dispatch / combine are used exactly as before."""

    def __init__(self, shape: fm.Shape, M: int, ids, w, mb_off, slot_expert, tok_src):
        self.real_shape, self.M, self.real_ids, self.real_slot_expert, self.tok_src = \
            shape, M, ids, slot_expert, tok_src
        sv = fm.virtual_shape(shape, M)
        dev = ids.device
        ids_v = torch.empty_like(ids)
        se_v = torch.empty(tuple(slot_expert.shape[:-1]) + (shape.S * M,), dtype=torch.int32, device=dev)
        super().__init__(sv, ids_v, w, mb_off, se_v)
        self.traffic = torch.empty((shape.n_mb, shape.L, M, M), dtype=torch.int32, device=dev)

    def plan(self, quota_in: Optional[torch.Tensor] = None) -> None:
        fm.source_ids(self.real_shape, self.M, self.real_ids, self.tok_src, self.ids, self.status)
        fm.local_placement(self.real_shape, self.M, self.real_slot_expert, self.slot_expert, self.status)
        super().plan(quota_in)
        fm.traffic(self.real_shape, self.M, self.quota, self.traffic)


DEFAULT_LADDER = ((0, 0), (2, 1), (1, 1), (1, 2), (1, 4), (0, 1))    # theta = inf, 2, 1, 1/2, 1/4, 0 as (num, den)


class TradeoffStepPlan(LocalStepPlan):
    """Per-source Stage 4 under F = a * L_max + b * C_max (Eq.(10); DESIGN.md reading
    39): every member of the threshold ladder is solved exactly for every instance (quotas only), the
    objective picks one per instance, and the pairs are assigned on the chosen member.  Attributes as
    LocalStepPlan, plus ``member`` [n_mb,L], ``F`` [n_members,n_mb,L]; ``slot_expert`` is the chosen
    virtual placement [n_mb,L,S*M] and the plan's shape carries ``placement_mb_stride = L*S*M``."""

    def __init__(self, shape: fm.Shape, M: int, a: int, b: int, ids, w, mb_off, slot_expert, tok_src,
                 ladder=DEFAULT_LADDER):
        import dataclasses
        super().__init__(shape, M, ids, w, mb_off, slot_expert, tok_src)
        dev, s, n = ids.device, shape, len(ladder)
        self.a, self.b, self.ladder = a, b, tuple(ladder)
        sv = self.shape
        self.shape = dataclasses.replace(sv, placement_mb_stride=sv.L * sv.S)      # one placement per instance
        self._dp = None
        i32 = dict(dtype=torch.int32, device=dev)
        self.se_v_k = torch.empty((n, s.n_mb, s.L, sv.S), **i32)
        self.quota_k = torch.empty((n, s.n_mb, s.L, sv.S), **i32)
        self.rank_load_k = torch.empty((n, s.n_mb, s.L, s.P), **i32)
        self.slot_off_k = torch.empty((s.n_mb, s.L, sv.S + 1), **i32)              # scratch, not kept per member
        self.traffic_k = torch.empty((n, s.n_mb, s.L, M, M), **i32)
        self.member = torch.empty((s.n_mb, s.L), **i32)
        self.F = torch.empty((n, s.n_mb, s.L), dtype=torch.int64, device=dev)
        self.quota_sel = torch.empty((s.n_mb, s.L, sv.S), **i32)
        self.slot_expert = torch.empty((s.n_mb, s.L, sv.S), **i32)
        self.workspace = torch.empty(fm.workspace_bytes(self.shape) + 16, dtype=torch.uint8, device=dev)

    def plan(self, quota_in: Optional[torch.Tensor] = None) -> None:
        assert quota_in is None
        fm.source_ids(self.real_shape, self.M, self.real_ids, self.tok_src, self.ids, self.status)
        self.load_hist()
        self._stage4()

    def _stage4(self) -> None:
        rs, M = self.real_shape, self.M
        for k, (num, den) in enumerate(self.ladder):
            fm.local_placement_theta(rs, M, num, den, self.hist, self.real_slot_expert, self.se_v_k[k], self.status)
            fm.assign(self.shape, self.ids, self.mb_off, self.hist, self.se_v_k[k], None, self.quota_k[k],
                      self.rank_load_k[k], self.slot_off_k, None, None, self.workspace, self.status)
            fm.traffic(rs, M, self.quota_k[k], self.traffic_k[k])
        fm.tradeoff_select(rs, M, self.a, self.b, self.rank_load_k, self.traffic_k, self.quota_k, self.se_v_k,
                           self.member, self.F, self.quota_sel, self.slot_expert)
        self.assign(self.quota_sel)
        fm.traffic(rs, M, self.quota, self.traffic)


class Alg2StepPlan(TradeoffStepPlan):
    """The paper's planner for the recompute stage, all on the device: Alg. 1 (Stage 1, machine + rank
    level) from the step totals, then per (micro-step, layer) Alg. 2 Stage 2 (relocation by swaps), Stage
    3 (replica search) and Stage 4 under the same objective F = a * L_max + b * C_max (
    DESIGN.md readings 33-35, 37, 39, 40).  ``slot_expert_mb`` [n_mb,L,S] is the per-instance placement
    of Stages 1-3; the plan's own ``slot_expert`` / ``quota`` / ``inv`` refer to the commodity instance
    as in TradeoffStepPlan."""

    def __init__(self, shape: fm.Shape, M: int, a: int, b: int, ids, w, mb_off, tok_src, win: int = 4,
                 max_rounds: int = 32, max_copies: int = 8, ladder=None):
        import dataclasses
        dev = ids.device
        if ladder is None:
            ladder = DEFAULT_LADDER if M > 1 else ((0, 1),)        # one machine: every member is the same
        base = torch.empty((shape.L, shape.S), dtype=torch.int32, device=dev)
        super().__init__(shape, M, a, b, ids, w, mb_off, base, tok_src, ladder)
        self.base_slot_expert = base
        self.win, self.max_rounds, self.max_copies = win, max_rounds, max_copies
        self.slot_expert_mb = torch.empty((shape.n_mb, shape.L, shape.S), dtype=torch.int32, device=dev)
        self.swaps = torch.empty((shape.n_mb, shape.L), dtype=torch.int32, device=dev)
        self.replicas = torch.empty((shape.n_mb, shape.L), dtype=torch.int32, device=dev)
        self.F_stage3 = torch.empty((shape.n_mb, shape.L, 2), dtype=torch.int64, device=dev)
        self.base_shape = shape
        # Stages 2-3 hand Stage 4 one placement per instance
        self.real_shape = dataclasses.replace(shape, placement_mb_stride=shape.L * shape.S)
        self.real_slot_expert = self.slot_expert_mb

    def plan(self, quota_in: Optional[torch.Tensor] = None) -> None:
        assert quota_in is None
        bs, M = self.base_shape, self.M
        fm.source_ids(bs, M, self.real_ids, self.tok_src, self.ids, self.status)
        self.load_hist()                                           # hist_v and its step totals
        fm.base_placement_machines(bs, M, self.a, self.b, self.step_hist, self.base_slot_expert, self.status)
        fm.swap_relocation(bs, M, self.win, self.max_rounds, self.a, self.b, self.hist, self.base_slot_expert,
                           self.slot_expert_mb, self.swaps, self.status)
        fm.replica_search(bs, M, self.max_copies, self.a, self.b, self.hist, self.slot_expert_mb,
                          self.slot_expert_mb, self.replicas, self.F_stage3, self.status)
        self._stage4()


class PlannerStepPlan(StepPlan):
    """All four planner stages on the device: Stage 1 (rank-level LPT from the step totals), Alg. 3
    Stages 2-3 per (micro-step, layer) over ``M`` machines, Stage 4 on the per-micro-step placements
    (PAPER.md:282-407, :787-846).  ``shape`` is the plain shape; the plan's own shape carries
    ``placement_mb_stride = L * S``."""

    def __init__(self, shape: fm.Shape, M: int, ids, w, mb_off):
        import dataclasses
        dev = ids.device
        self.M = M
        self.base_shape = shape
        self.base_slot_expert = torch.empty((shape.L, shape.S), dtype=torch.int32, device=dev)
        se_mb = torch.empty((shape.n_mb, shape.L, shape.S), dtype=torch.int32, device=dev)
        super().__init__(dataclasses.replace(shape, placement_mb_stride=shape.L * shape.S), ids, w, mb_off, se_mb)

    def plan(self, quota_in: Optional[torch.Tensor] = None) -> None:
        self.load_hist()
        fm.base_placement(self.base_shape, self.step_hist, self.base_slot_expert, self.status)
        fm.microstep_placement(self.base_shape, self.M, self.hist, self.base_slot_expert, self.slot_expert,
                               self.status)
        self.assign(quota_in)
