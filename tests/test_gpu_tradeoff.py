"""GPU parity of the per-source Stage 4 under F = a*L_max + b*C_max (foremoe_local_placement_theta,
quota-only foremoe_assign, foremoe_traffic, foremoe_tradeoff_select; runner.TradeoffStepPlan) against
oracle O15, bit-exact; and a HiGHS solution of Eq.(10) (the C rows included),
rounded to integers, fed through quota_in on the virtual shape."""
import math

import numpy as np
import pytest
import torch

from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import binding as fm
from paper_2606_11867_b200 import runner, synth
from tests import gpu_common as G
from tests.test_gpu_local import per_source_counts

pytestmark = pytest.mark.gpu


def tradeoff_plan(shape, M, a, b, ids, w, mb_off, se, tok_src):
    t = lambda x, dt: torch.as_tensor(np.ascontiguousarray(x), dtype=dt).to(G.DEV)
    tp = runner.TradeoffStepPlan(shape, M, a, b, t(ids, torch.int32), t(w, torch.float32), t(mb_off, torch.int32),
                                 t(se, torch.int32), t(tok_src, torch.int32))
    for name in ("quota", "rank_load", "slot_off", "pair_slot", "inv", "traffic", "member", "quota_sel", "slot_expert"):
        getattr(tp, name).fill_(-77)
    tp.plan()
    torch.cuda.synchronize()
    return tp


@pytest.mark.parametrize("cfg_id,kw,M,a,b", [
    (1, {}, 2, 1, 1),
    (2, dict(L=2, n_samples=12, sample_len=700, H=256, mb_samples=4), 2, 1, 1),
    (2, dict(L=2, n_samples=12, sample_len=700, H=256, mb_samples=4), 2, 1, 0),
    (2, dict(L=1, n_samples=8, sample_len=500, H=128, mb_samples=4), 4, 2, 5),
    (3, dict(L=1, n_samples=4, sample_len=1100, H=256, mb_samples=2), 8, 1, 2),
    (5, dict(L=1, n_samples=2, sample_len=3000, H=256, mb_samples=1), 4, 3, 1),
])
def test_tradeoff_plan_equals_oracle(cuda_device, cfg_id, kw, M, a, b):
    cfg = synth.config(cfg_id).scaled(**kw) if kw else synth.config(cfg_id)
    ids, w, mb_off, se = G.make_case(cfg)
    tok_src = synth.gen_tok_src(cfg)
    R = cfg.P // M
    tp = tradeoff_plan(fm.shape_of(cfg), M, a, b, ids, w, mb_off, se, tok_src)
    assert tp.faults() == 0
    ids_v = (ids.astype(np.int64) * M + (tok_src // R)[None, :, None]).astype(np.int32)
    members = []
    for l in range(cfg.L):
        for i in range(cfg.n_mb):
            a0, b0 = int(mb_off[i]), int(mb_off[i + 1])
            w_se = per_source_counts(ids[l, a0:b0], tok_src[a0:b0], cfg.P, cfg.E)
            ref = orc.quota_tradeoff(w_se, se[l], cfg.P, cfg.Ns, M, a, b)
            assert ref["fault"] == 0
            assert tp.F[:, i, l].cpu().numpy().tolist() == ref["F"].tolist(), ("F", l, i)
            assert int(tp.member[i, l]) == ref["member"], ("member", l, i)
            members.append(ref["member"])
            assert (tp.slot_expert[i, l].cpu().numpy() == ref["se_v"]).all(), ("se_v", l, i)
            assert (tp.quota[i, l].cpu().numpy() == ref["quota_v"]).all(), ("quota_v", l, i)
            assert (tp.rank_load[i, l].cpu().numpy() == ref["rank_load"]).all(), ("rank_load", l, i)
            assert (tp.slot_off[i, l].cpu().numpy() == ref["slot_off_v"]).all(), ("slot_off_v", l, i)
            assert (tp.traffic[i, l].cpu().numpy() == ref["traffic"]).all(), ("traffic", l, i)
            ps, inv, perm, f = orc.assign_instance(ids_v[l, a0:b0], ref["se_v"], ref["quota_v"], ref["slot_off_v"],
                                                   cfg.E * M, base=a0 * cfg.K)
            assert f == 0
            assert (tp.pair_slot[l, a0:b0].cpu().numpy().ravel() == ps).all(), ("pair_slot", l, i)
            assert (tp.inv[l, a0:b0].cpu().numpy().ravel() == inv).all(), ("inv", l, i)
    # the data path runs unchanged on the chosen plan
    l, i = 0, 0
    a0, b0 = int(mb_off[i]), int(mb_off[i + 1])
    n = b0 - a0
    x = synth.gen_activations(cfg, n, i, G.DEV)
    perm_g = torch.empty((n * cfg.K,), dtype=torch.int32, device=G.DEV)
    buf = torch.empty((n * cfg.K, cfg.H), dtype=tp.shape.act_torch_dtype, device=G.DEV)
    tp.dispatch(l, i, i + 1, x, perm_g, buf)
    inv0 = tp.inv[l, a0:b0].cpu().numpy()
    G.check_combine_random(tp, inv0, w[l, a0:b0], l, i, a0, n, seed=3, what="tradeoff")
    tok = (perm_g.long() - a0 * cfg.K) // cfg.K
    assert torch.equal(buf.view(torch.uint8), x.index_select(0, tok).view(torch.uint8))
    print(f"cfg{cfg_id} M={M} a={a} b={b}: members chosen {np.bincount(members, minlength=6).tolist()}")


def test_b0_reaches_the_unrestricted_optimum_and_big_b_stays_local(cuda_device):
    cfg = synth.config(2).scaled(L=2, n_samples=16, sample_len=600, H=128, mb_samples=4)
    M = 2
    ids, w, mb_off, se = G.make_case(cfg)
    tok_src = synth.gen_tok_src(cfg)
    shape = fm.shape_of(cfg)
    plain = G.gpu_plan(shape, ids, w, mb_off, se)                       # single-source Stage 4: min L_max
    t0 = tradeoff_plan(shape, M, 1, 0, ids, w, mb_off, se, tok_src)
    assert torch.equal(t0.rank_load.max(-1).values, plain.rank_load.max(-1).values)
    from tests.test_gpu_local import local_plan
    hard = local_plan(shape, M, ids, w, mb_off, se, tok_src)
    tb = tradeoff_plan(shape, M, 0, 1, ids, w, mb_off, se, tok_src)      # only C_max counts
    off = lambda tr: (tr - torch.diag_embed(torch.diagonal(tr, dim1=-2, dim2=-1))).amax((-1, -2))
    assert (off(tb.traffic) <= off(hard.traffic)).all()
    tm = tradeoff_plan(shape, M, 1, 1, ids, w, mb_off, se, tok_src)
    F = lambda p: p.rank_load.max(-1).values.long() + off(p.traffic).long()
    assert (F(tm) <= F(hard)).all() and (F(tm) <= F(t0)).all()


def _lp_eq10_solution(w_se, se, P, Ns, M, a, b):
    """HiGHS on Eq.(10) as printed (every copy allowed, L_r <= L*, C_ij <= C*): the fractional
    per-commodity split x[(e, m)][host slot] and the optimum value."""
    from scipy.optimize import linprog
    from tests import helpers as Hh
    R, E = P // M, w_se.shape[1]
    com = [(e, m, int(w_se[m * R:(m + 1) * R, e].sum())) for e in range(E) for m in range(M)]
    com = [c for c in com if c[2] > 0]
    hosts = {e: Hh.hosts_of(se, Ns, e) for e in range(E)}
    var = [(ci, j) for ci, (e, m, _) in enumerate(com) for j in hosts[e]]
    nv = len(var)
    cost = np.zeros(nv + 2)
    cost[nv], cost[nv + 1] = a, b
    A_eq = np.zeros((len(com), nv + 2))
    A_ub = np.zeros((P + M * M, nv + 2))
    for v, (ci, j) in enumerate(var):
        A_eq[ci, v] = 1.0
        A_ub[j // Ns, v] = 1.0
        if com[ci][1] != (j // Ns) // R:
            A_ub[P + com[ci][1] * M + (j // Ns) // R, v] = 1.0
    A_ub[:P, nv] = -1.0
    A_ub[P:, nv + 1] = -1.0
    res = linprog(cost, A_ub=A_ub, b_ub=np.zeros(P + M * M), A_eq=A_eq, b_eq=np.array([c[2] for c in com], float),
                  bounds=[(0, None)] * (nv + 2), method="highs")
    assert res.status == 0
    return com, var, res.x[:nv], float(res.fun)


def test_lp_solution_fed_through_quota_in(cuda_device):
    """The paper's own Stage 4: Eq.(10) solved by HiGHS on the host, its fractional
    split rounded to whole tokens per commodity (largest remainder, ties to the lowest slot) and handed
    to foremoe_assign as quota_in on the VIRTUAL shape (every copy allowed).  The device validates
    Eq.(8)/(9), lays the pairs out, and the resulting loads / traffic stay within the rounding slack of
    the LP optimum; the oracle given the same quota_in agrees bit for bit."""
    cfg = synth.config(2).scaled(L=1, n_samples=8, sample_len=600, H=128, mb_samples=4)
    M, a, b = 2, 1, 1
    R = cfg.P // M
    ids, w, mb_off, se = G.make_case(cfg)
    tok_src = synth.gen_tok_src(cfg)
    shape = fm.shape_of(cfg)
    sv = fm.virtual_shape(shape, M)
    t = lambda x, dt: torch.as_tensor(np.ascontiguousarray(x), dtype=dt).to(G.DEV)
    ids_v = (ids.astype(np.int64) * M + (tok_src // R)[None, :, None]).astype(np.int32)
    # every copy allowed for every source machine: theta = 0 member (num = 0, den = 1)
    hist_v, _, f = orc.load_hist(ids_v, mb_off, cfg.E * M)
    qin = np.zeros((cfg.n_mb, cfg.L, cfg.S * M), dtype=np.int32)
    se_v = np.zeros((cfg.n_mb, cfg.L, cfg.S * M), dtype=np.int32)
    lp_val = np.zeros((cfg.n_mb, cfg.L))
    n_com = np.zeros((cfg.n_mb, cfg.L), dtype=np.int64)
    for l in range(cfg.L):
        for i in range(cfg.n_mb):
            a0, b0 = int(mb_off[i]), int(mb_off[i + 1])
            w_se = per_source_counts(ids[l, a0:b0], tok_src[a0:b0], cfg.P, cfg.E)
            se_v[i, l], f = orc.local_placement_theta(hist_v[i, l], se[l], cfg.E, cfg.P, cfg.Ns, M, 0, 1)
            assert f == 0
            com, var, x, lp_val[i, l] = _lp_eq10_solution(w_se, se[l], cfg.P, cfg.Ns, M, a, b)
            n_com[i, l] = len(com)
            for ci, (e, m, cnt) in enumerate(com):        # largest-remainder rounding per commodity
                idx = [v for v, (c2, _) in enumerate(var) if c2 == ci]
                frac = np.clip(x[idx], 0, None)
                base = np.floor(frac + 1e-9).astype(np.int64)
                rem = cnt - int(base.sum())
                order = sorted(range(len(idx)), key=lambda k: (-(frac[k] - base[k]), var[idx[k]][1]))
                for k in order[:rem]:
                    base[k] += 1
                for k, v in enumerate(idx):
                    qin[i, l, var[v][1] * M + m] = base[k]
    import dataclasses
    sv_mb = dataclasses.replace(sv, placement_mb_stride=sv.L * sv.S)
    sp = runner.StepPlan(sv_mb, t(ids_v, torch.int32), t(w, torch.float32), t(mb_off, torch.int32), t(se_v, torch.int32))
    sp.plan(t(qin, torch.int32))
    torch.cuda.synchronize()
    assert sp.faults() == 0                                   # Eq.(8)/(9) hold for the rounded LP solution
    assert (sp.quota.cpu().numpy() == qin).all()
    traffic = torch.empty((cfg.n_mb, cfg.L, M, M), dtype=torch.int32, device=G.DEV)
    fm.traffic(shape, M, sp.quota, traffic)
    tr = traffic.cpu().numpy().astype(np.int64)
    for l in range(cfg.L):
        for i in range(cfg.n_mb):
            a0, b0 = int(mb_off[i]), int(mb_off[i + 1])
            off = tr[i, l].copy()
            np.fill_diagonal(off, 0)
            F = a * int(sp.rank_load[i, l].max()) + b * int(off.max())
            # rounding moves at most one token per (commodity, host): F within (a + b) * #commodities of LP*
            assert lp_val[i, l] - 1e-6 <= F <= lp_val[i, l] + (a + b) * n_com[i, l]
            q, so = qin[i, l], np.concatenate([[0], np.cumsum(qin[i, l])]).astype(np.int32)
            ps, inv, perm, f = orc.assign_instance(ids_v[l, a0:b0], se_v[i, l], q, so, cfg.E * M, base=a0 * cfg.K)
            assert f == 0
            assert (sp.pair_slot[l, a0:b0].cpu().numpy().ravel() == ps).all()
            assert (sp.inv[l, a0:b0].cpu().numpy().ravel() == inv).all()
    # and the ladder's own answer for the same instances is not far from the LP either (reported)
    tp = tradeoff_plan(shape, M, a, b, ids, w, mb_off, se, tok_src)
    Fsel = tp.F.gather(0, tp.member.long()[None]).squeeze(0).cpu().numpy().astype(float)
    print("ladder F / LP*: mean %.4f max %.4f" % (float((Fsel / lp_val).mean()), float((Fsel / lp_val).max())))


@pytest.mark.parametrize("cfg_id,kw,M,a,b", [
    (2, dict(L=2, n_samples=12, sample_len=700, H=256, mb_samples=4), 2, 1, 1),
    (2, dict(L=1, n_samples=8, sample_len=500, H=128, mb_samples=4), 1, 1, 0),
    (3, dict(L=1, n_samples=4, sample_len=1100, H=256, mb_samples=2), 8, 1, 2),
])
def test_alg2_planner_chain_equals_oracle_chain(cuda_device, cfg_id, kw, M, a, b):
    """runner.Alg2StepPlan (Alg. 1 -> swaps -> replica search -> Stage 4 under a*L_max + b*C_max, all on
    the device) against the same chain of oracles O14 -> O12 -> O16 -> O15, stage by stage."""
    cfg = synth.config(cfg_id).scaled(**kw)
    ids, w, mb_off, _ = G.make_case(cfg)
    tok_src = synth.gen_tok_src(cfg)
    R = cfg.P // M
    t = lambda x, dt: torch.as_tensor(np.ascontiguousarray(x), dtype=dt).to(G.DEV)
    ap = runner.Alg2StepPlan(fm.shape_of(cfg), M, a, b, t(ids, torch.int32), t(w, torch.float32), t(mb_off, torch.int32),
                             t(tok_src, torch.int32))
    ap.plan()
    torch.cuda.synchronize()
    assert ap.faults() == 0
    ladder = ap.ladder
    for l in range(cfg.L):
        # per-source-machine loads of every instance and of the step
        c_me = np.zeros((cfg.n_mb, M, cfg.E), dtype=np.int64)
        for i in range(cfg.n_mb):
            a0, b0 = int(mb_off[i]), int(mb_off[i + 1])
            w_se = per_source_counts(ids[l, a0:b0], tok_src[a0:b0], cfg.P, cfg.E)
            c_me[i] = w_se.reshape(M, R, cfg.E).sum(1)
        base, f = orc.base_placement_machines(c_me.sum(0), cfg.P, cfg.Nb, cfg.Nr, M, a, b)
        assert f == 0 and (ap.base_slot_expert[l].cpu().numpy() == base).all(), ("stage 1", l)
        for i in range(cfg.n_mb):
            a0, b0 = int(mb_off[i]), int(mb_off[i + 1])
            sw, st, f = orc.swap_relocation(c_me[i].astype(np.int32), base, cfg.P, cfg.Nb, cfg.Nr, M, ap.win,
                                            ap.max_rounds, a, b)
            assert f == 0 and int(ap.swaps[i, l]) == st[0]
            rs, st3, f = orc.replica_search(c_me[i].astype(np.int32), sw, cfg.P, cfg.Nb, cfg.Nr, M, a, b,
                                            max_copies=ap.max_copies)
            assert f == 0 and (ap.slot_expert_mb[i, l].cpu().numpy() == rs).all(), ("stages 2-3", l, i)
            assert int(ap.replicas[i, l]) == st3[0] and ap.F_stage3[i, l].tolist() == [int(st3[1]), int(st3[2])]
            w_se = per_source_counts(ids[l, a0:b0], tok_src[a0:b0], cfg.P, cfg.E)
            ref = orc.quota_tradeoff(w_se, rs, cfg.P, cfg.Ns, M, a, b, ladder=ladder)
            assert ref["fault"] == 0 and int(ap.member[i, l]) == ref["member"]
            assert (ap.quota[i, l].cpu().numpy() == ref["quota_v"]).all(), ("stage 4", l, i)
            assert (ap.traffic[i, l].cpu().numpy() == ref["traffic"]).all()
            ids_v = (ids[l, a0:b0].astype(np.int64) * M + (tok_src[a0:b0] // R)[:, None]).astype(np.int32)
            ps, inv, perm, f = orc.assign_instance(ids_v, ref["se_v"], ref["quota_v"], ref["slot_off_v"], cfg.E * M,
                                                   base=a0 * cfg.K)
            assert f == 0 and (ap.inv[l, a0:b0].cpu().numpy().ravel() == inv).all()


def test_theta_spill_rule_with_products_beyond_64_bits(cuda_device):
    """The spill test of a ladder member, c * den * P > num * n_loc * total (include/foremoe.h,
    foremoe_local_placement_theta), with P = 16 384 ranks, counts near 2^30 and theta = 2^20 / 2^20: both
    sides pass 2^63.  Expected placement from the rule itself in Python's unbounded integers."""
    P, Nb, Nr, M = 16384, 1, 1, 2
    E, Ns, S, R = P * Nb, Nb + Nr, P * (Nb + Nr), P // M
    rng = np.random.default_rng(77)
    shape = fm.Shape(L=1, E=E, K=1, P=P, Nb=Nb, Nr=Nr, T=8, n_mb=1, H=8, act_dtype=fm.ACT_FP32)
    se = np.full((P, Ns), -1, dtype=np.int32)
    se[:, 0] = rng.permutation(E)
    se[:, 1] = rng.integers(-1, E, size=P)                  # replicas anywhere (some on the other machine)
    se = se.reshape(1, S)
    hv = rng.integers(0, 50, size=(E, M)).astype(np.int64)
    big = rng.choice(E, size=E // 2, replace=False)
    hv[big] = rng.integers(1 << 29, (1 << 30) + 1, size=(E // 2, M))      # half of the experts carry almost everything
    num, den = (1 << 20) - 3, 1 << 20
    total = int(hv.sum())
    assert total * num > 1 << 63 and int(hv.max()) * den * P > 1 << 63
    # rule in exact integers: n_loc(e, m) = ranks of machine m holding e
    holds = [[set() for _ in range(M)] for _ in range(E)]
    for j in range(S):
        e = int(se[0, j])
        if e >= 0:
            holds[e][(j // Ns) // R].add(j // Ns)
    exp = np.full(S * M, -1, dtype=np.int32)
    n_spill = 0
    for j in range(S):
        e = int(se[0, j])
        if e < 0:
            continue
        for m in range(M):
            n = len(holds[e][m])
            spill = n > 0 and int(hv[e, m]) * den * P > num * n * total
            n_spill += bool(spill and (j // Ns) // R != m)
            if (j // Ns) // R == m or n == 0 or spill:
                exp[j * M + m] = e * M + m
    assert n_spill > 0
    dev = G.DEV
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    out = torch.full((1, 1, S * M), -7, dtype=torch.int32, device=dev)
    fm.local_placement_theta(shape, M, num, den, torch.as_tensor(hv.astype(np.int32)).reshape(1, 1, E * M).to(dev),
                             torch.as_tensor(se).to(dev), out, st)
    torch.cuda.synchronize()
    assert int(st.item()) == 0
    got = out.cpu().numpy().ravel()
    assert (got == exp).all(), np.argwhere(got != exp)[:5].tolist()
