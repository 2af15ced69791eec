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
    q = None if quota_in is None else t(quota_in, torch.int32)
    sp.plan(q)                                   # foremoe_plan: two passes over the ids
    torch.cuda.synchronize()
    # foremoe_load_hist + foremoe_assign (three passes) must give the same bits in every output
    names = ("hist", "step_hist", "quota", "rank_load", "slot_off", "pair_slot", "inv")
    fused = {n: getattr(sp, n).clone() for n in names}
    f_fused = sp.faults()
    for n in names:
        getattr(sp, n).fill_(-77)
    sp.status.zero_()
    sp.load_hist()
    sp.assign(q)
    torch.cuda.synchronize()
    assert sp.faults() == f_fused
    for n in names:                              # (deterministic on faulted inputs as well)
        assert torch.equal(fused[n], getattr(sp, n)), ("foremoe_plan vs load_hist + assign", n)
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
            # the combine is defined on the experts' OUTPUTS, which differ per k:
            # with expert_out = buf the K rows of a token are identical and a w_k <-> row mix-up
            # would go unseen, so every instance is also combined on independent random rows
            check_combine_random(sp, ref["inv"][l, a:b], w_h[l, a:b], l, i, a, n,
                                 seed=1000 * l + i, what=what)
    return worst


def random_expert_out(n_rows: int, H: int, dtype, seed: int) -> torch.Tensor:
    """Independent random rows in slot order (a stand-in for the experts' outputs): N(0,1) with a
    few large / tiny / negative-zero values so that a wrong row, weight or order shows in the bits."""
    g = torch.Generator(device=DEV).manual_seed(seed)
    eo = torch.randn((max(n_rows, 1), H), generator=g, device=DEV)
    u = torch.rand((max(n_rows, 1), H), generator=g, device=DEV)
    eo = torch.where(u < 0.01, eo * 1e4, eo)
    eo = torch.where(u > 0.99, eo * 1e-4, eo)
    eo = torch.where((u > 0.5) & (u < 0.505), torch.full_like(eo, -0.0), eo)
    return eo.to(dtype).contiguous()


def check_combine_random(sp: runner.StepPlan, inv_ref, w_ref, l: int, i: int, a: int, n: int,
                         seed: int, what: str = "", mb_end=None, eo=None):
    """foremoe_combine of micro-steps [i, mb_end) of layer l on random expert outputs against O6,
    bit for bit.  inv_ref / w_ref: the oracle's inv and the weights of tokens [a, a+n)."""
    s = sp.shape
    if n == 0:
        return
    if eo is None:
        eo = random_expert_out(n * s.K, s.H, s.act_torch_dtype, seed)
    y = torch.full((n, s.H), float("nan"), dtype=torch.float32, device=DEV)
    sp.combine(l, i, i + 1 if mb_end is None else mb_end, eo, y)
    torch.cuda.synchronize()
    y_ref = orc.combine(np.asarray(inv_ref).reshape(n, s.K), np.asarray(w_ref).reshape(n, s.K),
                        to_bits(eo)[:n * s.K], s.act_dtype, row_base=a * s.K)
    y_g = y.cpu().numpy()
    bad = np.argwhere(y_g.view(np.uint32) != y_ref.view(np.uint32))
    assert bad.size == 0, f"{what} combine(random expert_out) l={l} mb={i}: {len(bad)} words differ, " \
                          f"first at {bad[0]}: gpu {y_g[tuple(bad[0])]} oracle {y_ref[tuple(bad[0])]}"


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


def random_case(rng, L, E, K, P, Nr, mb_sizes, dup_tokens=False, empty_slots=True,
                 same_rank_dup=True, skew=1.0):
    Nb = E // P
    Ns = Nb + Nr
    S = P * Ns
    T = int(sum(mb_sizes))
    mb_off = np.concatenate([[0], np.cumsum(mb_sizes)]).astype(np.int32)
    p = (np.arange(E) + 1.0) ** (-skew)
    p /= p.sum()
    ids = np.empty((L, T, K), dtype=np.int32)
    for l in range(L):
        perm = rng.permutation(E)
        if dup_tokens:
            ids[l] = perm[rng.choice(E, size=(T, K), p=p)]
        else:
            g = rng.gumbel(size=(T, E)) + np.log(p)[None, :]
            ids[l] = perm[np.argsort(-g, axis=1)[:, :K]]
    w = rng.random((L, T, K), dtype=np.float32)
    se = np.full((L, S), -1, dtype=np.int32)
    for l in range(L):
        base = rng.permutation(E)
        for r in range(P):
            se[l, r * Ns:r * Ns + Nb] = base[r * Nb:(r + 1) * Nb]
            for a in range(Nr):
                u = rng.random()
                if empty_slots and u < 0.2:
                    continue
                if same_rank_dup and u < 0.35:
                    se[l, r * Ns + Nb + a] = se[l, r * Ns + rng.integers(Nb)]   # inactive duplicate
                else:
                    se[l, r * Ns + Nb + a] = rng.integers(E)
    return ids, w, mb_off, se, Nb, Ns
