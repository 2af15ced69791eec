"""Helpers of the GPU parity tests: run the CUDA path through the C-ABI binding and the oracle on
the same arrays, and compare element by element."""
from __future__ import annotations

import numpy as np
import torch

from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import binding as fm
from paper_2606_11867_b200 import runner, synth

DEV = "cuda:0"


def to_bits(t: torch.Tensor) -> np.ndarray:
    """Host numpy view of activations: uint16 bit patterns for bf16, float32 otherwise."""
    t = t.detach().cpu().contiguous()
    if t.dtype == torch.bfloat16:
        return t.view(torch.int16).numpy().view(np.uint16)
    return t.numpy()


def oracle_plan(ids, mb_off, se, E, P, Ns, quota_in=None):
    hist, step, f1 = orc.load_hist(ids, mb_off, E)
    plan = orc.plan(ids, mb_off, hist, se, P, Ns, quota_in=quota_in)
    plan["hist"], plan["step_hist"] = hist, step
    plan["fault"] |= f1
    return plan


def gpu_plan(shape: fm.Shape, ids, w, mb_off, se, quota_in=None) -> runner.StepPlan:
    t = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).to(DEV)
    sp = runner.StepPlan(shape, t(ids, torch.int32), t(w, torch.float32), t(mb_off, torch.int32),
                         t(se, torch.int32))
    # poison the outputs so that unwritten elements are caught
    for name in ("hist", "quota", "rank_load", "slot_off", "pair_slot", "inv"):
        getattr(sp, name).fill_(-77)
    sp.plan(None if quota_in is None else t(quota_in, torch.int32))
    torch.cuda.synchronize()
    return sp


def assert_plan_equal(sp: runner.StepPlan, ref: dict, what: str = ""):
    for name in ("hist", "step_hist", "quota", "rank_load", "slot_off", "pair_slot", "inv"):
        got = getattr(sp, name).cpu().numpy()
        exp = ref[name]
        assert got.shape == exp.shape, (what, name, got.shape, exp.shape)
        bad = np.argwhere(got != exp)
        assert bad.size == 0, f"{what} {name}: {len(bad)} mismatches, first at {bad[0]}: " \
                              f"gpu {got[tuple(bad[0])]} oracle {exp[tuple(bad[0])]}"


def check_data_path(sp: runner.StepPlan, ref: dict, x_by_mb, layers, mbs, what: str = ""):
    """dispatch + combine of the given instances against O5 / O6, bit for bit (perm, buf) and
    within 1e-6 max relative error (y; the same fma order makes it bit-identical in practice)."""
    s = sp.shape
    mb_off = sp.mb_off.cpu().numpy()
    w_h = sp.w.cpu().numpy()
    worst = 0.0
    for l in layers:
        for i in mbs:
            a, b = int(mb_off[i]), int(mb_off[i + 1])
            n = b - a
            x = x_by_mb[i]
            perm = torch.full((max(n * s.K, 1),), -5, dtype=torch.int32, device=DEV)
            buf = torch.empty((max(n * s.K, 1), s.H), dtype=s.act_torch_dtype, device=DEV)
            y = torch.empty((max(n, 1), s.H), dtype=torch.float32, device=DEV)
            buf.view(torch.uint8).fill_(0xAB)
            y.fill_(float("nan"))
            sp.dispatch(l, i, i + 1, x, perm, buf)
            sp.combine(l, i, i + 1, buf, y)
            torch.cuda.synchronize()
            if n == 0:
                continue
            perm_ref = ref["perm"][l, a * s.K:b * s.K]
            assert (perm[:n * s.K].cpu().numpy() == perm_ref).all(), (what, "perm", l, i)
            xb = to_bits(x)
            buf_ref = orc.gather(perm_ref, xb, s.K, pair_base=a * s.K)
            assert (to_bits(buf)[:n * s.K] == buf_ref).all(), (what, "buf", l, i)
            y_ref = orc.combine(ref["inv"][l, a:b], w_h[l, a:b], buf_ref, s.act_dtype,
                                row_base=a * s.K)
            y_g = y[:n].cpu().numpy()
            rel = np.abs(y_g - y_ref) / np.maximum(np.abs(y_ref), 1e-30)
            worst = max(worst, float(rel.max()))
            assert rel.max() <= 1e-6, (what, "y", l, i, float(rel.max()))
            assert (y_g.view(np.uint32) == y_ref.view(np.uint32)).all(), (what, "y bits", l, i)
    return worst


def make_case(cfg: synth.TraceConfig, device: str = "cpu"):
    ids, w, mb_off = synth.gen_trace(cfg, device)
    ids, w, mb_off = ids.cpu().numpy(), w.cpu().numpy(), mb_off.cpu().numpy()
    hist, step, fault = orc.load_hist(ids, mb_off, cfg.E)
    assert fault == 0
    se = synth.gen_placement(cfg, step)
    return ids, w, mb_off, se


def activations(cfg: synth.TraceConfig, mb_off, mbs):
    return {i: synth.gen_activations(cfg, max(int(mb_off[i + 1] - mb_off[i]), 1), i, DEV)
            for i in mbs}
