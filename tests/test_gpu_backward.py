"""GPU parity of the backward data path (foremoe_combine_bwd / foremoe_dispatch_bwd) against the
oracle (O9 / O10): gradient rows bit-exact (the bf16 rounding decision is taken on the same fp32
product on both sides), dx bit-identical (same fp32 add order), dw within the derived bound
H * 2^-24 * sum_h |dy * eo| of the exactly accumulated oracle value (reading 28).
"""
import dataclasses

import numpy as np
import pytest
import torch

from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import binding as fm
from paper_2606_11867_b200 import synth
from tests import gpu_common as G

pytestmark = pytest.mark.gpu


def _rows(shape, n_rows, seed, scale=1.0):
    g = torch.Generator(device="cpu").manual_seed(seed)
    t = (torch.randn((max(n_rows, 1), shape.H), generator=g) * scale).to(shape.act_torch_dtype)
    return t.to(G.DEV)


def _float_rows(bits, act_dtype):
    if act_dtype == 0:
        return torch.from_numpy(bits.view(np.int16).copy()).view(torch.bfloat16).float().numpy()
    return bits


def check_backward(sp, ref, layers, mbs, what="", want_dw=True):
    s = sp.shape
    mb_off = sp.mb_off.cpu().numpy()
    w_h = sp.w.cpu().numpy()
    dw = torch.full((s.L, s.T, s.K), float("nan"), dtype=torch.float32, device=G.DEV) if want_dw else None
    worst_dw = 0.0
    for l in layers:
        for i in mbs:
            a, b = int(mb_off[i]), int(mb_off[i + 1])
            n = b - a
            eo = _rows(s, n * s.K, 1000 + 17 * l + i)
            g = torch.Generator(device="cpu").manual_seed(2000 + 17 * l + i)
            dy = torch.randn((max(n, 1), s.H), generator=g).to(G.DEV)
            d_eo = torch.empty_like(eo)
            d_eo.view(torch.uint8).fill_(0xAB)
            dx = torch.full((max(n, 1), s.H), float("nan"), dtype=torch.float32, device=G.DEV)
            sp.combine_bwd(l, i, i + 1, dy, eo if want_dw else None, d_eo, dw)
            sp.dispatch_bwd(l, i, i + 1, d_eo, dx)
            torch.cuda.synchronize()
            if n == 0:
                continue
            inv = ref["inv"][l, a:b]
            eo_b, dy_h = G.to_bits(eo)[:n * s.K], dy[:n].cpu().numpy()
            init = np.full((n * s.K, s.H), 0xABAB if s.act_dtype == 0 else 0, dtype=eo_b.dtype)
            if s.act_dtype == 1:
                init = np.frombuffer(bytes([0xAB]) * (n * s.K * s.H * 4), dtype=np.float32).reshape(n * s.K, s.H)
            d_ref, dw_ref = orc.combine_bwd(inv, w_h[l, a:b], dy_h, eo_b if want_dw else None, s.act_dtype,
                                            n * s.K, row_base=a * s.K, d_eo_init=init)
            got = G.to_bits(d_eo)[:n * s.K]
            assert (got.view(np.uint8) == d_ref.view(np.uint8)).all(), (what, "d_eo", l, i)
            dx_ref = orc.dispatch_bwd(inv, d_ref, s.act_dtype, row_base=a * s.K)
            ok_tok = (inv >= 0).all(1)              # tokens with a skipped pair read an untouched row
            assert (dx[:n].cpu().numpy().view(np.uint32)[ok_tok] == dx_ref.view(np.uint32)[ok_tok]).all(), (what, "dx", l, i)
            if want_dw:
                dw_g = dw[l, a:b].cpu().numpy()
                v = _float_rows(eo_b, s.act_dtype).astype(np.float64)
                safe = np.where(inv >= 0, inv - a * s.K, 0)
                bound = s.H * 2.0 ** -24 * np.einsum("th,tkh->tk", np.abs(dy_h.astype(np.float64)), np.abs(v[safe]))
                err = np.abs(dw_g.astype(np.float64) - dw_ref)
                assert (err <= bound + 1e-30).all(), (what, "dw", l, i, float((err / (bound + 1e-30)).max()))
                worst_dw = max(worst_dw, float((err / (bound + 1e-30)).max()))
    return worst_dw


def _case(cfg):
    ids, w, mb_off, se = G.make_case(cfg)
    ref = G.oracle_plan(ids, mb_off, se, cfg.E, cfg.P, cfg.Ns)
    sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se)
    assert ref["fault"] == 0 and sp.faults() == 0
    return sp, ref


def test_tiny_config1_backward(cuda_device):
    """Config 1 (fp32 rows, K = 2), every instance."""
    cfg = synth.config(1)
    sp, ref = _case(cfg)
    check_backward(sp, ref, range(cfg.L), range(cfg.n_mb), "cfg1")
    check_backward(sp, ref, [0], [0, cfg.n_mb - 1], "cfg1-no-dw", want_dw=False)


@pytest.mark.parametrize("cfg_id,kw", [
    (2, dict(L=2, n_samples=12, sample_len=700, H=2048, mb_samples=4)),   # K=8, several slices per row
    (3, dict(L=1, n_samples=4, sample_len=900, H=7168, mb_samples=2)),    # 28 slices per row
    (5, dict(L=1, n_samples=2, sample_len=2500, H=4096, mb_samples=1)),   # K=10
    (4, dict(L=1, n_samples=9, H=512, mb_samples=2)),                     # ragged micro-steps, 2 slices
])
def test_scaled_configs_backward(cuda_device, cfg_id, kw):
    cfg = synth.config(cfg_id).scaled(**kw)
    sp, ref = _case(cfg)
    r = check_backward(sp, ref, range(cfg.L), range(cfg.n_mb), f"cfg{cfg_id}-scaled")
    assert r < 0.25          # observed dw error sits far inside the worst-case bound
    check_backward(sp, ref, [cfg.L - 1], [0], f"cfg{cfg_id}-scaled-no-dw", want_dw=False)


@pytest.mark.parametrize("K,H,bf16", [(1, 8, False), (3, 40, True), (5, 264, True), (32, 72, False),
                                      (7, 1000, True), (4, 520, True), (6, 136, False)])
def test_generic_k_and_ragged_rows(cuda_device, K, H, bf16):
    """K outside the specialised set (generic kernel), rows that are not a multiple of 512 bytes,
    empty micro-steps."""
    rng = np.random.default_rng(K * 100 + H)
    P, Nb, Nr, L = 4, 8, 1, 2
    E = P * Nb
    sizes = [0, 77, 130, 0, 301]
    T = sum(sizes)
    mb_off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int32)
    ids = np.stack([np.stack([rng.permutation(E)[:K] for _ in range(T)]) for _ in range(L)]).astype(np.int32)
    w = rng.standard_normal((L, T, K)).astype(np.float32)
    shape = fm.Shape(L=L, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=T, n_mb=len(sizes), H=H,
                     act_dtype=fm.ACT_BF16 if bf16 else fm.ACT_FP32)
    se = np.full((L, P * (Nb + Nr)), -1, dtype=np.int32)
    for l in range(L):
        pe = rng.permutation(E)
        for r in range(P):
            se[l, r * (Nb + Nr):r * (Nb + Nr) + Nb] = pe[r * Nb:(r + 1) * Nb]
            se[l, r * (Nb + Nr) + Nb] = pe[(r * Nb + Nb) % E]          # a replica of another rank's expert
    ref = G.oracle_plan(ids, mb_off, se, E, P, Nb + Nr)
    sp = G.gpu_plan(shape, ids, w, mb_off, se)
    assert ref["fault"] == 0 and sp.faults() == 0
    G.assert_plan_equal(sp, ref, "generic")
    check_backward(sp, ref, range(L), range(len(sizes)), f"K{K}-H{H}")


def test_ranged_backward_and_unit_weight_identity(cuda_device):
    """A ranged call over several micro-steps equals the per-instance calls; dispatch_bwd equals
    combine with unit weights bit for bit; backward of the identity expert: dx = (sum_k w) * dy
    up to the rounding of the gradient rows."""
    cfg = synth.config(2).scaled(L=2, n_samples=10, sample_len=333, H=256, mb_samples=3)
    sp, ref = _case(cfg)
    s = sp.shape
    mb_off = sp.mb_off.cpu().numpy()
    l, (b, e) = 1, (1, 4)
    a_tok, b_tok = int(mb_off[b]), int(mb_off[e])
    n = b_tok - a_tok
    eo = _rows(s, n * s.K, 5)
    dy = torch.randn((n, s.H), generator=torch.Generator().manual_seed(6)).to(G.DEV)
    d1 = torch.zeros_like(eo)
    d2 = torch.zeros_like(eo)
    dw1 = torch.zeros((s.L, s.T, s.K), dtype=torch.float32, device=G.DEV)
    dw2 = torch.zeros_like(dw1)
    sp.combine_bwd(l, b, e, dy, eo, d1, dw1)
    for i in range(b, e):
        r0, r1 = (int(mb_off[i]) - a_tok), (int(mb_off[i + 1]) - a_tok)
        sp.combine_bwd(l, i, i + 1, dy[r0:r1], eo[r0 * s.K:r1 * s.K], d2[r0 * s.K:r1 * s.K], dw2)
    dx = torch.empty((n, s.H), dtype=torch.float32, device=G.DEV)
    y1 = torch.empty_like(dx)
    sp.dispatch_bwd(l, b, e, d1, dx)
    fm.combine(s, l, b, e, sp.mb_off, sp.inv, torch.ones_like(sp.w), d1, y1)
    torch.cuda.synchronize()
    assert torch.equal(d1.view(torch.int16), d2.view(torch.int16)) and torch.equal(dw1, dw2)
    assert torch.equal(dx.view(torch.int32), y1.view(torch.int32))
    wsum = sp.w[l, a_tok:b_tok].sum(1, keepdim=True)
    assert torch.allclose(dx, wsum * dy, rtol=2 ** -7, atol=1e-3)


def test_backward_host_errors(cuda_device):
    cfg = synth.config(1)
    sp, ref = _case(cfg)
    s = sp.shape
    n = cfg.T // cfg.n_mb
    eo = _rows(s, n * s.K, 1)
    dy = torch.zeros((n, s.H), device=G.DEV)
    d = torch.zeros_like(eo)
    dw = torch.zeros((s.L, s.T, s.K), device=G.DEV)
    for kw in (dict(layer=s.L), dict(mb_begin=-1), dict(mb_end=s.n_mb + 1), dict(mb_begin=2, mb_end=1)):
        a = dict(layer=0, mb_begin=0, mb_end=1)
        a.update(kw)
        with pytest.raises(fm.ForeMoEError):
            fm.combine_bwd(s, a["layer"], a["mb_begin"], a["mb_end"], sp.mb_off, sp.inv, sp.w, dy, eo, d, dw)
        with pytest.raises(fm.ForeMoEError):
            fm.dispatch_bwd(s, a["layer"], a["mb_begin"], a["mb_end"], sp.mb_off, sp.inv, d, dy)
    with pytest.raises(fm.ForeMoEError):                      # dw without the forward expert outputs
        fm.combine_bwd(s, 0, 0, 1, sp.mb_off, sp.inv, sp.w, dy, None, d, dw)
    with pytest.raises(fm.ForeMoEError):                      # misaligned rows
        fm.combine_bwd(s, 0, 0, 1, sp.mb_off, sp.inv, sp.w, dy, eo, d.view(-1)[1:], None)


@pytest.mark.parametrize("cfg_id", [1, 2])
def test_backward_skips_faulted_pairs(cuda_device, cfg_id):
    """Pairs with an invalid expert id get inv = -1 in the plan (fault ID_RANGE): the backward leaves
    the rows no pair maps to untouched, writes dw = 0 for them and sums only the valid rows into dx
    (fp32 rows: K = 2; bf16 rows: K = 8 with several slices per row)."""
    cfg = synth.config(1) if cfg_id == 1 else synth.config(2).scaled(L=1, n_samples=4, sample_len=300, H=1024, mb_samples=2)
    ids, w, mb_off, se = G.make_case(cfg)
    bad = ids.copy()
    bad[0, 3, 1] = cfg.E + 3
    bad[0, 40, 0] = -1
    bad[0, int(mb_off[1]) + 7, cfg.K - 1] = 1 << 20
    ref = G.oracle_plan(bad, mb_off, se, cfg.E, cfg.P, cfg.Ns)
    sp = G.gpu_plan(fm.shape_of(cfg), bad, w, mb_off, se)
    assert sp.faults() == fm.FAULT_ID_RANGE and ref["fault"] == orc.FAULT_ID_RANGE
    G.assert_plan_equal(sp, ref, "bad-id")
    assert (ref["inv"][0] < 0).sum() == 3
    check_backward(sp, ref, [0], [0, 1], "bad-id-bwd")
    # the skipped tokens too: dx sums the rows that exist (rows of d_eo the oracle and the GPU agree on)
    s = sp.shape
    a, b = 0, int(mb_off[1])
    eo = _rows(s, b * s.K, 77)
    dy = torch.randn((b, s.H), generator=torch.Generator().manual_seed(78)).to(G.DEV)
    d_eo = torch.zeros_like(eo)
    dw = torch.full((s.L, s.T, s.K), float("nan"), dtype=torch.float32, device=G.DEV)
    dx = torch.empty((b, s.H), dtype=torch.float32, device=G.DEV)
    sp.combine_bwd(0, 0, 1, dy, eo, d_eo, dw)
    sp.dispatch_bwd(0, 0, 1, d_eo, dx)
    torch.cuda.synchronize()
    inv = ref["inv"][0, a:b]
    d_ref, dw_ref = orc.combine_bwd(inv, w[0, a:b], dy.cpu().numpy(), G.to_bits(eo), s.act_dtype, b * s.K)
    assert (G.to_bits(d_eo) == d_ref).all()
    assert (dx.cpu().numpy().view(np.uint32) == orc.dispatch_bwd(inv, d_ref, s.act_dtype).view(np.uint32)).all()
    dw_g = dw[0, a:b].cpu().numpy()
    assert (dw_g[inv < 0] == 0).all() and (dw_ref[inv < 0] == 0).all()
