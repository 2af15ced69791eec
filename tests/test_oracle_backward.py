"""Pins for oracle O9 (combine backward = MoE dispatch of gradients) and O10 (dispatch backward =
MoE combine of gradients), sec. 7.1 (n1 = 3, n2 = 4) and :170 (same plan as forward).

Pinned against things other than the oracle: torch.autograd on a float64 forward built from
index_select / einsum (library routine), the adjoint identities of the two linear maps, torch's
own bf16 conversion plus hand-picked rounding ties, closed forms.
"""
import numpy as np
import pytest
import torch

from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import synth


def _bits(x: torch.Tensor) -> np.ndarray:
    return x.view(torch.int16).numpy().view(np.uint16)


def _from_bits(b: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(b.view(np.int16).copy()).view(torch.bfloat16)


@pytest.fixture(scope="module")
def case():
    """One instance of a reduced config-2 trace: inv, w of micro-step 1, layer 1."""
    cfg = synth.config(2).scaled(L=2, n_samples=6, sample_len=300, H=96, mb_samples=2)
    ids, w, mb_off = synth.gen_trace(cfg, "cpu")
    ids, w, mb_off = ids.numpy(), w.numpy(), mb_off.numpy()
    hist, step, fault = orc.load_hist(ids, mb_off, cfg.E)
    se = synth.gen_placement(cfg, step)
    plan = orc.plan(ids, mb_off, hist, se, cfg.P, cfg.Ns)
    assert fault == 0 and plan["fault"] == 0
    i, l = 1, 1
    a, b = int(mb_off[i]), int(mb_off[i + 1])
    return cfg, plan["inv"][l][a:b].copy(), w[l, a:b].copy(), a * cfg.K, b - a


def _autograd(inv_local, w, eo64, x64, dy64, K):
    """float64 forward with library ops; returns (d_eo, dw, dx) from torch.autograd."""
    n, H = x64.shape
    inv_t = torch.from_numpy(inv_local.astype(np.int64))
    # forward dispatch: buf[inv[t,k]] = x[t]  <=>  buf = x[perm // K]
    perm = torch.empty(n * K, dtype=torch.int64)
    perm[inv_t.reshape(-1)] = torch.arange(n * K)
    x = x64.clone().requires_grad_(True)
    buf = x.index_select(0, perm // K)
    eo = eo64.clone().requires_grad_(True)
    wt = torch.from_numpy(w.astype(np.float64)).requires_grad_(True)
    y = torch.einsum("tk,tkh->th", wt, eo.index_select(0, inv_t.reshape(-1)).reshape(n, K, H))
    d_eo, dw = torch.autograd.grad((y * dy64).sum(), (eo, wt))
    g_buf = d_eo                      # gradient arriving at buf when the expert is the identity
    (dx,) = torch.autograd.grad((buf * g_buf).sum(), (x,))
    return d_eo.numpy(), dw.numpy(), dx.numpy()


def test_backward_vs_autograd_fp32_rows(case):
    cfg, inv, w, base, n = case
    K, H = cfg.K, cfg.H
    rng = np.random.default_rng(1)
    eo = rng.standard_normal((n * K, H)).astype(np.float32)
    dy = rng.standard_normal((n, H)).astype(np.float32)
    x = rng.standard_normal((n, H)).astype(np.float32)
    d_eo, dw = orc.combine_bwd(inv, w, dy, eo, 1, n * K, row_base=base)
    ref_deo, ref_dw, ref_dx = _autograd(inv - base, w, torch.from_numpy(eo).double(),
                                   torch.from_numpy(x).double(), torch.from_numpy(dy).double(), K)
    # d_eo: one fp32 multiply per element -> within half an ulp of the exact product
    assert (np.abs(d_eo - ref_deo) <= 2.0 ** -24 * np.abs(ref_deo) + 1e-45).all()
    # dw: fp64 accumulation rounded once
    assert (np.abs(dw - ref_dw) <= 2.0 ** -23 * np.abs(ref_dw) + 1e-30).all()
    # dx from the gradient rows (fp32 adds, k ascending): K-term sum bound
    dx = orc.dispatch_bwd(inv, d_eo, 1, row_base=base)
    g = d_eo.astype(np.float64)[inv - base]                       # [n, K, H]
    assert (np.abs(dx - g.sum(1)) <= K * 2.0 ** -24 * np.abs(g).sum(1) + 1e-30).all()
    # the same through autograd of the gather (the transpose of index_select), fed with the exact d_eo
    assert (np.abs(dx - ref_dx) <= (K + 1) * 2.0 ** -24 * np.abs(ref_deo[inv - base]).sum(1) + 1e-30).all()
    # a wrong index (rows of another pair) must not pass
    inv_bad = np.roll(inv, 1, axis=1)
    d_bad, dw_bad = orc.combine_bwd(inv_bad, w, dy, eo, 1, n * K, row_base=base)
    assert not np.allclose(d_bad, ref_deo, rtol=1e-3) and not np.allclose(dw_bad, ref_dw, rtol=1e-3, atol=1e-3)


def test_adjoint_identities(case):
    """<C(eo), dy> = <eo, C^T dy> and <D x, g> = <x, D^T g>, with forward C = O6, D = O5."""
    cfg, inv, w, base, n = case
    K, H = cfg.K, cfg.H
    rng = np.random.default_rng(2)
    eo = rng.standard_normal((n * K, H)).astype(np.float32)
    dy = rng.standard_normal((n, H)).astype(np.float32)
    x = rng.standard_normal((n, H)).astype(np.float32)
    g = rng.standard_normal((n * K, H)).astype(np.float32)
    y = orc.combine(inv, w, eo, 1, row_base=base)
    d_eo, _ = orc.combine_bwd(inv, w, dy, eo, 1, n * K, row_base=base)
    lhs = (y.astype(np.float64) * dy).sum()
    rhs = (eo.astype(np.float64) * d_eo).sum()
    scale = (np.abs(eo.astype(np.float64)) * np.abs(d_eo)).sum()
    assert abs(lhs - rhs) <= 1e-6 * scale
    perm = np.empty(n * K, dtype=np.int32)
    perm[(inv - base).ravel()] = np.arange(n * K, dtype=np.int32) + base
    buf = orc.gather(perm, x, K, pair_base=base)
    dx = orc.dispatch_bwd(inv, g, 1, row_base=base)
    lhs = (buf.astype(np.float64) * g).sum()
    rhs = (x.astype(np.float64) * dx).sum()
    assert abs(lhs - rhs) <= 1e-6 * (np.abs(x.astype(np.float64)) * np.abs(dx)).sum()


def test_dw_is_directional_derivative(case):
    """y is linear in w: <C(eo, w + d) - C(eo, w), dy> = <dw, d> (checked in float64 via O6 on
    exactly representable small integers, so the forward has no rounding at all)."""
    cfg, inv, w, base, n = case
    K, H = cfg.K, cfg.H
    rng = np.random.default_rng(3)
    eo = rng.integers(-8, 9, size=(n * K, H)).astype(np.float32)
    dy = rng.integers(-4, 5, size=(n, H)).astype(np.float32)
    w0 = rng.integers(-3, 4, size=(n, K)).astype(np.float32)
    dlt = rng.integers(-2, 3, size=(n, K)).astype(np.float32)
    y0 = orc.combine(inv, w0, eo, 1, row_base=base)
    y1 = orc.combine(inv, w0 + dlt, eo, 1, row_base=base)
    _, dw = orc.combine_bwd(inv, w0, dy, eo, 1, n * K, row_base=base)
    lhs = ((y1.astype(np.float64) - y0) * dy).sum()
    assert lhs == (dw.astype(np.float64) * dlt).sum()             # all integers: exact


def test_bf16_rows_rounding(case):
    cfg, inv, w, base, n = case
    K, H = cfg.K, cfg.H
    rng = np.random.default_rng(4)
    dy = rng.standard_normal((n, H)).astype(np.float32)
    eo = torch.from_numpy(rng.standard_normal((n * K, H)).astype(np.float32)).bfloat16()
    d_eo, dw = orc.combine_bwd(inv, w, dy, _bits(eo), 0, n * K, row_base=base)
    # the fp32 product, then torch's round-to-nearest-even conversion (library routine)
    prod = torch.from_numpy(w)[:, :, None] * torch.from_numpy(dy)[:, None, :]      # fp32 [n,K,H]
    ref = torch.empty((n * K, H), dtype=torch.bfloat16)
    ref[torch.from_numpy((inv - base).astype(np.int64)).reshape(-1)] = prod.reshape(n * K, H).bfloat16()
    assert (d_eo == _bits(ref)).all()
    ref_dw = (dy.astype(np.float64)[:, None, :] * eo.float().numpy().astype(np.float64)[inv - base]).sum(-1)
    assert (np.abs(dw - ref_dw) <= 2.0 ** -23 * np.abs(ref_dw) + 1e-30).all()
    # dx of bf16 gradient rows
    dx = orc.dispatch_bwd(inv, d_eo, 0, row_base=base)
    gg = _from_bits(d_eo).float().numpy().astype(np.float64)[inv - base]
    assert (np.abs(dx - gg.sum(1)) <= K * 2.0 ** -24 * np.abs(gg).sum(1) + 1e-30).all()


def test_bf16_rounding_ties_by_hand():
    """w * dy values chosen on and around rounding ties of the 8-bit bf16 significand."""
    inv = np.array([[0], [1], [2], [3], [4], [5]], dtype=np.int32)
    w = np.ones((6, 1), dtype=np.float32)
    dy = np.array([[1.0 + 2.0 ** -8],              # tie, even below      -> 1.0
                   [1.0 + 2.0 ** -7 + 2.0 ** -8],  # tie, odd below       -> 1 + 2^-6
                   [1.0 + 2.0 ** -8 + 2.0 ** -20], # just above the tie   -> 1 + 2^-7
                   [-(1.0 + 2.0 ** -8)],           # sign symmetric       -> -1.0
                   [2.0 ** -133],                  # subnormal bf16, exact (a multiple of 2^-133)
                   [3.3895313892515355e38]],       # 0x7F7F0000 bf16 max: stays finite
                  dtype=np.float32)
    d_eo, _ = orc.combine_bwd(inv, w, dy, None, 0, 6)
    got = _from_bits(d_eo).float().numpy().ravel()
    assert got.tolist() == [1.0, 1.0 + 2.0 ** -6, 1.0 + 2.0 ** -7, -1.0, 2.0 ** -133, 3.3895313892515355e38]
    # and the product itself is rounded to fp32 BEFORE the bf16 decision (two roundings, reading 27):
    # w = 1 + 2^-12, dy = 1 + 2^-12 + 2^-23: exact product 1 + 2^-11 + 2^-23 + 2^-24 + ..., fp32 keeps it
    w2 = np.array([[np.float32(1 + 2.0 ** -12)]], dtype=np.float32)
    dy2 = np.array([[np.float32(1 + 2.0 ** -12)]], dtype=np.float32)
    d2, _ = orc.combine_bwd(np.array([[0]], np.int32), w2, dy2, None, 0, 1)
    assert _from_bits(d2).float().item() == torch.tensor(float(w2[0, 0] * dy2[0, 0])).bfloat16().float().item()


def test_closed_forms_and_skipped_pairs():
    K, H, n = 3, 8, 4
    inv = np.arange(n * K, dtype=np.int32).reshape(n, K)[:, ::-1].copy()
    inv[2, 1] = -1                                                # a faulted pair: skipped
    w = np.full((n, K), 0.5, dtype=np.float32)
    dy = np.ones((n, H), dtype=np.float32)
    eo = np.arange(n * K * H, dtype=np.float32).reshape(n * K, H)
    init = np.full((n * K, H), 7.0, dtype=np.float32)
    d_eo, dw = orc.combine_bwd(inv, w, dy, eo, 1, n * K, d_eo_init=init)
    hit = np.zeros(n * K, dtype=bool)
    hit[inv[inv >= 0]] = True
    assert (d_eo[hit] == 0.5).all() and (d_eo[~hit] == 7.0).all() and (~hit).sum() == 1
    for t in range(n):
        for k in range(K):
            exp = 0.0 if inv[t, k] < 0 else eo[inv[t, k]].sum()   # dy = 1: dw = row sum
            assert dw[t, k] == exp
    dx = orc.dispatch_bwd(inv, np.ones((n * K, H), np.float32), 1)
    assert (dx[[0, 1, 3]] == K).all() and (dx[2] == K - 1).all()
    # O10 equals O6 with unit weights (definition: fma(1, v, acc) = acc + v exactly)
    inv_ok = np.arange(n * K, dtype=np.int32).reshape(n, K)
    g = np.random.default_rng(0).standard_normal((n * K, H)).astype(np.float32)
    assert (orc.dispatch_bwd(inv_ok, g, 1) == orc.combine(inv_ok, np.ones((n, K), np.float32), g, 1)).all()
