"""Pins for oracle O1 (histogram), O3/O4 (pair->slot, stable counting sort), O5 (gather) and
O6 (combine): library routines, closed forms, invariants, exact special cases.
PAPER.md:204/:247 (w_{s,e}), :58 (dispatch/combine), :56 (weighted sum), Eq.(8)/(9) :266-270.
"""
import numpy as np
import pytest
import torch

from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import synth


def _trace(cfg):
    ids, w, mb_off = synth.gen_trace(cfg, "cpu")
    return ids.numpy(), w.numpy(), mb_off.numpy()


@pytest.fixture(scope="module")
def tiny():
    cfg = synth.config(1)
    ids, w, mb_off = _trace(cfg)
    hist, step, fault = orc.load_hist(ids, mb_off, cfg.E)
    assert fault == 0
    se = synth.gen_placement(cfg, step)
    plan = orc.plan(ids, mb_off, hist, se, cfg.P, cfg.Ns)
    assert plan["fault"] == 0
    return cfg, ids, w, mb_off, hist, step, se, plan


@pytest.fixture(scope="module")
def qwen_small():
    cfg = synth.config(2).scaled(L=2, n_samples=12, sample_len=700, H=512, mb_samples=4)
    ids, w, mb_off = _trace(cfg)
    hist, step, fault = orc.load_hist(ids, mb_off, cfg.E)
    assert fault == 0
    se = synth.gen_placement(cfg, step)
    plan = orc.plan(ids, mb_off, hist, se, cfg.P, cfg.Ns)
    assert plan["fault"] == 0
    return cfg, ids, w, mb_off, hist, step, se, plan


# ------------------------------------------------------------------ O1
def test_hist_bincount(tiny, qwen_small):
    for cfg, ids, w, mb_off, hist, step, se, plan in (tiny, qwen_small):
        for i in range(cfg.n_mb):
            a, b = mb_off[i], mb_off[i + 1]
            for l in range(cfg.L):
                ref = np.bincount(ids[l, a:b].ravel(), minlength=cfg.E)
                assert (hist[i, l] == ref).all()
                assert hist[i, l].sum() == (b - a) * cfg.K       # histogram sums equal T*k
        assert (step == hist.sum(axis=0)).all()


def test_hist_closed_form():
    L, T, K, E = 2, 96, 4, 8
    p = np.arange(T * K).reshape(T, K)
    ids = np.stack([(p % E), ((p // 3) % E)]).astype(np.int32)
    mb_off = np.array([0, 32, 32, 96], dtype=np.int32)       # one empty micro-step
    hist, step, fault = orc.load_hist(ids, mb_off, E)
    assert fault == 0
    assert (hist[0, 0] == 32 * K // E).all() and (hist[1] == 0).all()
    assert (hist[2, 0] == 64 * K // E).all()
    assert step[0].tolist() == [T * K // E] * E
    assert hist[:, 1].sum() == T * K


def test_hist_faults():
    ids = np.zeros((1, 4, 2), dtype=np.int32)
    ids[0, 1, 1] = 9
    _, _, fault = orc.load_hist(ids, np.array([0, 4], dtype=np.int32), 8)
    assert fault == orc.FAULT_ID_RANGE
    _, _, fault = orc.load_hist(ids, np.array([0, 3], dtype=np.int32), 16)
    assert fault == orc.FAULT_MB_OFF
    _, _, fault = orc.load_hist(ids, np.array([0, 3, 2, 4], dtype=np.int32), 16)
    assert fault == orc.FAULT_MB_OFF


# ------------------------------------------------------------------ O3 / O4
def test_assign_pins(tiny, qwen_small):
    for cfg, ids, w, mb_off, hist, step, se, plan in (tiny, qwen_small):
        K, S = cfg.K, cfg.S
        for l in range(cfg.L):
            for i in range(cfg.n_mb):
                a, b = int(mb_off[i]) * K, int(mb_off[i + 1]) * K
                e = ids[l].reshape(-1)[a:b]
                ps = plan["pair_slot"][l].reshape(-1)[a:b]
                inv = plan["inv"][l].reshape(-1)[a:b]
                perm = plan["perm"][l][a:b]
                q = plan["quota"][i, l]
                so = plan["slot_off"][i, l]
                # every token lands on a slot hosting its expert (Eq.(9))
                assert (se[l][ps] == e).all()
                # per-slot pair counts equal the quotas; per-rank loads equal their quota sums
                cnt = np.bincount(ps, minlength=S)
                assert (cnt == q).all()
                assert (cnt.reshape(cfg.P, cfg.Ns).sum(1) == plan["rank_load"][i, l]).all()
                assert (so == np.concatenate([[0], np.cumsum(cnt)])).all()
                # stable counting sort == numpy's stable argsort (layer-global indices)
                assert (perm - a == np.argsort(ps, kind="stable")).all()
                # bijection, inverse
                assert (np.sort(perm) == np.arange(a, b)).all()
                assert (perm[inv - a] == np.arange(a, b)).all()
                # stable: strictly increasing inside every slot
                for j in range(S):
                    seg = perm[so[j]:so[j + 1]]
                    assert (np.diff(seg) > 0).all()
                # O3: contiguous blocks of the expert's stable order, replicas ascending
                for ex in np.unique(e):
                    slots_seq = ps[e == ex]
                    assert (np.diff(slots_seq) >= 0).all()


def test_assign_brute_force_tiny():
    """T <= 6: any per-token assignment meeting the quotas has the same rank loads; the oracle's
    is the one that hands contiguous blocks of token order to ascending replicas."""
    E, K = 3, 1
    se = np.array([0, 1, 2, 0], dtype=np.int32)          # P=2, Ns=2: expert 0 on both ranks
    ids = np.array([0, 1, 0, 0, 2, 0], dtype=np.int32)
    c = np.bincount(ids, minlength=E).astype(np.int32)
    q, rl, so, _, fault = orc.quota(c, se, 2, 2)
    assert fault == 0 and rl.tolist() == [3, 3] and q.tolist() == [2, 1, 1, 2]
    ps, inv, perm, fault = orc.assign_instance(ids, se, q, so, E, base=100)
    assert fault == 0
    assert ps.tolist() == [0, 1, 0, 3, 2, 3]
    assert inv.tolist() == [100, 102, 101, 104, 103, 105]
    assert perm.tolist() == [100, 102, 101, 104, 103, 105]


# ------------------------------------------------------------------ O5
def test_gather_pin(tiny, qwen_small):
    for cfg, ids, w, mb_off, hist, step, se, plan in (tiny, qwen_small):
        K = cfg.K
        i, l = cfg.n_mb - 1, cfg.L - 1
        a, b = int(mb_off[i]), int(mb_off[i + 1])
        x = synth.gen_activations(cfg, b - a, tag=i)
        xn = x.view(torch.int16).numpy().view(np.uint16) if cfg.act_dtype == 0 else x.numpy()
        perm = plan["perm"][l][a * K:b * K]
        buf = orc.gather(perm, xn, K, pair_base=a * K)
        assert (buf == xn[(perm - a * K) // K]).all()
        # every row in slot j belongs to a token that selected slot_expert[j]
        so = plan["slot_off"][i, l]
        rows = np.searchsorted(so, np.arange((b - a) * K), side="right") - 1
        tok = (perm - a * K) // K
        for d in range(0, (b - a) * K, 97):
            assert se[l][rows[d]] in ids[l, a + tok[d]]


# ------------------------------------------------------------------ O6
def _bits(x):
    return x.view(torch.int16).numpy().view(np.uint16)


def test_combine_exact_cases(tiny, qwen_small):
    """combine(dispatch(x)) with unit weights reproduces K*x exactly; w = 1/K reproduces x."""
    for cfg, ids, w, mb_off, hist, step, se, plan in (tiny, qwen_small):
        K = cfg.K
        i, l = 0, 0
        a, b = int(mb_off[i]), int(mb_off[i + 1])
        x = synth.gen_activations(cfg, b - a, tag=i)
        xn = _bits(x) if cfg.act_dtype == 0 else x.numpy()
        perm = plan["perm"][l][a * K:b * K]
        inv = plan["inv"][l][a:b]
        buf = orc.gather(perm, xn, K, pair_base=a * K)
        xf = x.float().numpy()
        y = orc.combine(inv, np.ones((b - a, K), np.float32), buf, cfg.act_dtype, row_base=a * K)
        assert (y == K * xf).all()
        y = orc.combine(inv, np.full((b - a, K), 1.0 / K, np.float32), buf, cfg.act_dtype,
                        row_base=a * K)
        assert (y == xf).all()


def test_combine_vs_float64(qwen_small):
    cfg, ids, w, mb_off, hist, step, se, plan = qwen_small
    K = cfg.K
    i, l = 1, 1
    a, b = int(mb_off[i]), int(mb_off[i + 1])
    rng = np.random.default_rng(5)
    # expert outputs differ per row (not the identity expert): catches a wrong row index
    eo = torch.from_numpy(rng.standard_normal(((b - a) * K, cfg.H)).astype(np.float32)).bfloat16()
    inv = plan["inv"][l][a:b]
    wi = w[l, a:b]
    y = orc.combine(inv, wi, _bits(eo), 0, row_base=a * K)
    v = eo.float().numpy().astype(np.float64)[inv - a * K]            # [n, K, H]
    ref = (wi.astype(np.float64)[:, :, None] * v).sum(1)
    bound = K * 2.0 ** -24 * (np.abs(wi.astype(np.float64))[:, :, None] * np.abs(v)).sum(1)
    assert (np.abs(y - ref) <= bound + 1e-30).all()
    # and it is not something else: a transposed weight order must fail the same bound
    y_bad = orc.combine(inv, wi[:, ::-1].copy(), _bits(eo), 0, row_base=a * K)
    assert not (np.abs(y_bad - ref) <= bound + 1e-30).all()


def test_combine_fixed_order_small():
    """fp32 fmaf chain, k ascending, from acc = 0: a case where the order matters."""
    inv = np.array([[0, 1, 2]], dtype=np.int32)
    w = np.array([[1.0, 1.0, 1.0]], dtype=np.float32)
    eo = np.array([[2.0 ** 24], [1.0], [-2.0 ** 24]], dtype=np.float32)
    y = orc.combine(inv, w, eo, 1)
    assert y[0, 0] == 0.0            # (2^24 + 1) rounds to 2^24 in fp32, then cancels
    y = orc.combine(np.array([[0, 2, 1]], dtype=np.int32), w, eo, 1)
    assert y[0, 0] == 1.0
    # fused multiply-add: w*v is not rounded before the add
    wv = np.float32(1.0 + 2.0 ** -12)
    eo2 = np.array([[wv], [-(np.float32(wv) * np.float32(wv))]], dtype=np.float32)
    y = orc.combine(np.array([[1, 0]], dtype=np.int32), np.array([[1.0, wv]], np.float32), eo2, 1)
    exact = float(wv) * float(wv) - float(np.float32(wv) * np.float32(wv))
    assert y[0, 0] == np.float32(exact) and exact != 0.0


def test_combine_skips_faulted_pairs():
    """A pair with inv < 0 has no dispatched row (foremoe.h; reading 38): it contributes nothing --
    the result equals the combine of the remaining pairs alone (same order), whatever the rows hold,
    and a token without any valid pair gives exactly 0."""
    rng = np.random.default_rng(8)
    n, K, H = 50, 4, 24
    eo = rng.standard_normal((n * K, H)).astype(np.float32)
    eo[7] = np.nan                                       # no pair maps here
    inv = rng.permutation(n * K).astype(np.int32).reshape(n, K)
    w = rng.random((n, K), dtype=np.float32)
    hit = np.argwhere(inv == 7)[0]
    inv[hit[0], hit[1]] = -1
    inv[3, :] = -1
    inv[5, 0] = -1
    inv[6, K - 1] = -1
    y = orc.combine(inv, w, eo, 1)
    assert np.isfinite(y).all() and (y[3] == 0).all()
    for t in range(n):
        keep = [k for k in range(K) if inv[t, k] >= 0]
        if not keep:
            continue
        y_t = orc.combine(inv[t:t + 1, keep], w[t:t + 1, keep], eo, 1)
        assert (y_t[0].view(np.uint32) == y[t].view(np.uint32)).all()
    # with a row base: layer-global rows, the -1 marker is not shifted
    y2 = orc.combine(np.where(inv >= 0, inv + 400, -1).astype(np.int32), w, eo, 1, row_base=400)
    assert (y2.view(np.uint32) == y.view(np.uint32)).all()


# ------------------------------------------------------------------ workload sanity (context)
def test_balance_improves_on_natural_placement(qwen_small):
    """Not parity: the synthetic trace is skewed, and the planned assignment is near-balanced
    (paper context: natural L_max/mean 2.5-5.8 -> ~1.02)."""
    cfg, ids, w, mb_off, hist, step, se, plan = qwen_small
    nat = synth.natural_placement(cfg)
    plan_nat = orc.plan(ids, mb_off, hist, nat, cfg.P, cfg.Ns)
    assert plan_nat["fault"] == 0
    r_nat = plan_nat["rank_load"].max(-1) / plan_nat["rank_load"].mean(-1)
    r_bal = plan["rank_load"].max(-1) / plan["rank_load"].mean(-1)
    assert r_nat.mean() > 1.2
    assert r_bal.mean() < r_nat.mean() and r_bal.mean() < 1.1
