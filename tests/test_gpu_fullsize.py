"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (the same
bench.Workload object, the same per-instance dispatch / combine calls).

The oracle cannot run a whole 1536-instance step in test time, so (tests/ rule of DESIGN.md sec. 5):
  * O1 histogram: every instance, every bin, against the oracle;
  * O2 quotas / rank loads / offsets and O3/O4 pair_slot / inv: every micro-step of layers
    {0, L/2, L-1} against the oracle, element by element;
  * O5 / O6 rows (perm, buf, y): layers {0, L/2, L-1} x micro-steps {first, last, most imbalanced}
    against the oracle, bit for bit;
  * every OTHER instance: properties that hold at any size, evaluated on the GPU with library
    routines (bincount, sort, cumsum, index_select): conservation Eq.(8), feasibility Eq.(9),
    offsets = prefix of quotas, rank loads = quota sums, inv is a bijection onto the instance's rows,
    per-slot pair counts = quotas, stability, and max rank load within the water-filling bound;
  * backward (O9 / O10): first and last instance against the oracle (gradient rows and dx bit for
    bit, dw within the derived bound), three random instances against torch library ops.
"""
import numpy as np
import pytest
import torch

import bench
from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import synth
from tests import gpu_common as G

pytestmark = pytest.mark.gpu


def _properties_all_instances(wl):
    """Invariants of the plan for EVERY instance, computed with torch library ops on the GPU."""
    sp, s = wl.plan, wl.shape
    dev = sp.ids.device
    mb = torch.from_numpy(wl.mb_off_h.astype(np.int64)).to(dev)
    tok = (mb[1:] - mb[:-1])
    se = sp.slot_expert.long()                                   # [L, S]
    quota = sp.quota.long()                                      # [n_mb, L, S]
    hist = sp.hist.long()
    assert (quota >= 0).all()
    # histogram sums equal T_i * K
    assert torch.equal(hist.sum(-1), (tok * s.K)[:, None].expand(-1, s.L))
    # Eq.(8) conservation / Eq.(9) feasibility: quotas of the slots holding e sum to c[e]; empty
    # slots get nothing
    per_e = torch.zeros((s.n_mb, s.L, s.E + 1), dtype=torch.int64, device=dev)
    idx = torch.where(se >= 0, se, torch.full_like(se, s.E))[None].expand(s.n_mb, -1, -1)
    per_e.scatter_add_(2, idx, quota)
    assert torch.equal(per_e[..., :s.E], hist) and (per_e[..., s.E] == 0).all()
    # offsets and rank loads
    so = sp.slot_off.long()
    assert (so[..., 0] == 0).all() and torch.equal(so[..., 1:], quota.cumsum(-1))
    assert torch.equal(sp.rank_load.long(), quota.view(s.n_mb, s.L, s.P, s.Ns).sum(-1))
    # the rule's quality: max rank load is optimal, hence <= ceil(mean) + (largest forced load
    # effects); a cheap universal bound: it never exceeds the natural (no-split) placement's max
    rl = sp.rank_load.long()
    assert (rl.sum(-1) == (tok * s.K)[:, None]).all()
    worst = 0.0
    for l in range(s.L):
        ids_l, ps_l, inv_l = sp.ids[l].long(), sp.pair_slot[l].long(), sp.inv[l].long()
        # every pair sits on a slot that hosts its expert
        assert torch.equal(se[l][ps_l.view(-1)], ids_l.view(-1))
        for i in range(s.n_mb):
            a, b = int(mb[i]) * s.K, int(mb[i + 1]) * s.K
            if a == b:
                continue
            ps, iv = ps_l.view(-1)[a:b], inv_l.view(-1)[a:b]
            # per-slot pair counts equal the quotas
            assert torch.equal(torch.bincount(ps, minlength=s.S), quota[i, l])
            # inv is a bijection onto the instance's rows [a, b)
            srt, order = torch.sort(iv)
            assert torch.equal(srt, torch.arange(a, b, device=dev))
            # rows are grouped by slot in ascending slot order and stable inside a slot:
            # walking rows in order, (slot, pair index) is strictly increasing lexicographically
            key = ps[order] * (b - a) + order
            assert (key[1:] > key[:-1]).all()
            mean = float(rl[i, l].sum()) / s.P
            worst = max(worst, float(rl[i, l].max()) / max(mean, 1.0))
    return worst


def _oracle_checks(wl, layers, data_mbs):
    sp, s, cfg = wl.plan, wl.shape, wl.cfg
    ids_h = sp.ids.cpu().numpy()
    mb = wl.mb_off_h
    # O1: every instance
    hist, step, f = orc.load_hist(ids_h, mb, s.E)
    assert f == 0
    assert (sp.hist.cpu().numpy() == hist).all()
    assert (sp.step_hist.cpu().numpy() == step).all()
    w_h = None
    for l in layers:
        se = wl.se_h[l]
        inv_l = sp.inv[l].cpu().numpy()
        ps_l = sp.pair_slot[l].cpu().numpy()
        for i in range(s.n_mb):
            a, b = int(mb[i]), int(mb[i + 1])
            q, rl, so, _, f = orc.quota(hist[i, l], se, s.P, s.Ns)
            assert f == 0
            assert (sp.quota[i, l].cpu().numpy() == q).all(), ("quota", l, i)
            assert (sp.rank_load[i, l].cpu().numpy() == rl).all(), ("rank_load", l, i)
            assert (sp.slot_off[i, l].cpu().numpy() == so).all(), ("slot_off", l, i)
            ps, inv, perm, f = orc.assign_instance(ids_h[l, a:b], se, q, so, s.E, base=a * s.K)
            assert f == 0
            assert (ps_l[a:b].ravel() == ps).all(), ("pair_slot", l, i)
            assert (inv_l[a:b].ravel() == inv).all(), ("inv", l, i)
            if i not in data_mbs:
                continue
            # O5 / O6 in the bench's launch configuration
            n = b - a
            x = wl.x[i]
            wl.buf.view(torch.uint8).fill_(0xAB)
            wl.y.fill_(float("nan"))
            wl.perm.fill_(-5)
            sp.dispatch(l, i, i + 1, x, wl.perm, wl.buf)
            sp.combine(l, i, i + 1, wl.buf, wl.y)
            torch.cuda.synchronize()
            assert (wl.perm[:n * s.K].cpu().numpy() == perm).all(), ("perm", l, i)
            buf_ref = orc.gather(perm, G.to_bits(x[:n]), s.K, pair_base=a * s.K)
            assert (G.to_bits(wl.buf[:n * s.K]) == buf_ref).all(), ("buf", l, i)
            if w_h is None or w_h[0] != l:
                w_h = (l, sp.w[l].cpu().numpy())
            y_ref = orc.combine(inv.reshape(n, s.K), w_h[1][a:b], buf_ref, s.act_dtype,
                                row_base=a * s.K)
            y_g = wl.y[:n].cpu().numpy()
            rel = np.abs(y_g - y_ref) / np.maximum(np.abs(y_ref), 1e-30)
            assert rel.max() <= 1e-6, ("y", l, i, float(rel.max()))
            assert (y_g.view(np.uint32) == y_ref.view(np.uint32)).all(), ("y bits", l, i)
            # non-identity expert: independent random rows per k, same launch configuration
            G.check_combine_random(sp, inv.reshape(n, s.K), w_h[1][a:b], l, i, a, n,
                                   seed=7000 + 100 * l + i, what=f"cfg{cfg.cfg_id}")


def _library_data_checks(wl, instances):
    """buf == x[perm // K] (torch.index_select) and y against an fp64 weighted sum, on the GPU."""
    sp, s = wl.plan, wl.shape
    mb = wl.mb_off_h
    for (l, i) in instances:
        a, b = int(mb[i]), int(mb[i + 1])
        n = b - a
        if n == 0:
            continue
        sp.dispatch(l, i, i + 1, wl.x[i], wl.perm, wl.buf)
        sp.combine(l, i, i + 1, wl.buf, wl.y)
        tok = (wl.perm[:n * s.K].long() - a * s.K) // s.K
        ref = wl.x[i].index_select(0, tok)
        assert torch.equal(wl.buf[:n * s.K].view(torch.int16 if s.act_dtype == 0 else torch.int32),
                           ref.view(torch.int16 if s.act_dtype == 0 else torch.int32))
        # y within K * 2^-24 * sum|w v| of the float64 sum (fp32 fma chain error bound), in chunks
        inv = (sp.inv[l, a:b].long() - a * s.K)
        w = sp.w[l, a:b].double()
        for c0 in range(0, n, 2048):
            c1 = min(n, c0 + 2048)
            rows = wl.buf[inv[c0:c1].reshape(-1)].double().view(c1 - c0, s.K, s.H)
            exact = (rows * w[c0:c1, :, None]).sum(1)
            bound = s.K * 2.0 ** -24 * (rows.abs() * w[c0:c1, :, None].abs()).sum(1) + 1e-30
            assert ((wl.y[c0:c1].double() - exact).abs() <= bound).all()


def _most_imbalanced_mb(wl, l):
    nat = wl.plan.hist[:, l].long().view(wl.shape.n_mb, wl.shape.P, wl.shape.Nb).sum(-1).float()
    return int((nat.max(-1).values / nat.mean(-1).clamp(min=1)).argmax())


@pytest.mark.parametrize("cfg_id", [2, 3, 5])
def test_full_config(cuda_device, cfg_id):
    cfg = synth.config(cfg_id)
    wl = bench.Workload(cfg, cuda_device)
    wl.plan.plan()
    torch.cuda.synchronize()
    assert wl.plan.faults() == 0
    worst = _properties_all_instances(wl)
    print(f"config {cfg_id}: worst L_max / L_mean over all instances = {worst:.4f}")
    # reported, not asserted: with the placement fixed at step level the optimum itself can sit far
    # above the mean when micro-step hot spots differ from step totals
    layers = sorted({0, cfg.L // 2, cfg.L - 1})
    data = {l: sorted({0, cfg.n_mb - 1, _most_imbalanced_mb(wl, l)}) for l in layers}
    for l in layers:
        _oracle_checks(wl, [l], data[l])
    rng = np.random.default_rng(cfg_id)
    inst = [wl.instances[k] for k in rng.choice(len(wl.instances), size=6, replace=False)]
    _library_data_checks(wl, inst)
    assert wl.plan.faults() == 0


@pytest.mark.parametrize("mb_samples", [1, 8, 64])
def test_config4_size_sweep(cuda_device, mb_samples):
    """Config 4: lognormal lengths, micro-step size 1 / 8 / 64 samples (the largest is > 2^31 bytes
    of dispatched rows per instance at full length: 64-bit row offsets)."""
    cfg = synth.config(4, mb_samples=mb_samples)
    wl = bench.Workload(cfg, cuda_device)
    wl.plan.plan()
    torch.cuda.synchronize()
    assert wl.plan.faults() == 0
    _properties_all_instances(wl)
    layers = [0, cfg.L - 1]
    for l in layers:
        _oracle_checks(wl, [l], sorted({0, cfg.n_mb - 1, _most_imbalanced_mb(wl, l)}))


def _backward_checks(wl, instances, oracle_instances):
    """Backward of the data path at full size in the bench's launch configuration (Workload with
    stage="update"): against the oracle (O9 / O10) on `oracle_instances`, against torch library
    ops on the GPU (fp32 product -> bf16 conversion, fp64 einsum, index_select) on `instances`."""
    sp, s = wl.plan, wl.shape
    mb = wl.mb_off_h
    bits = torch.int16 if s.act_dtype == 0 else torch.int32
    for (l, i) in instances:
        a, b = int(mb[i]), int(mb[i + 1])
        n = b - a
        if n == 0:
            continue
        sp.dispatch(l, i, i + 1, wl.x[i], wl.perm, wl.buf)
        wl.d_buf.view(torch.uint8).fill_(0xAB)
        sp.combine_bwd(l, i, i + 1, wl.dy, wl.buf, wl.d_buf, wl.dw)
        sp.dispatch_bwd(l, i, i + 1, wl.d_buf, wl.dx)
        torch.cuda.synchronize()
        inv = (sp.inv[l, a:b].long() - a * s.K)                       # [n, K] local rows
        w = sp.w[l, a:b]
        for c0 in range(0, n, 2048):
            c1 = min(n, c0 + 2048)
            rows = inv[c0:c1].reshape(-1)
            prod = (w[c0:c1, :, None] * wl.dy[c0:c1, None, :]).to(s.act_torch_dtype)    # fp32 multiply, RNE
            assert torch.equal(wl.d_buf[rows].view(bits), prod.view(-1, s.H).view(bits)), ("d_eo", l, i)
            eo = wl.buf[rows].double().view(c1 - c0, s.K, s.H)
            dyd = wl.dy[c0:c1].double()
            exact = torch.einsum("th,tkh->tk", dyd, eo)
            bound = s.H * 2.0 ** -24 * torch.einsum("th,tkh->tk", dyd.abs(), eo.abs()) + 1e-30
            assert ((wl.dw[l, a + c0:a + c1].double() - exact).abs() <= bound).all(), ("dw", l, i)
            g = wl.d_buf[rows].double().view(c1 - c0, s.K, s.H)
            bnd = s.K * 2.0 ** -24 * g.abs().sum(1) + 1e-30
            assert ((wl.dx[c0:c1].double() - g.sum(1)).abs() <= bnd).all(), ("dx", l, i)
        if (l, i) in oracle_instances:
            inv_h = sp.inv[l, a:b].cpu().numpy()
            d_ref, dw_ref = orc.combine_bwd(inv_h, w.cpu().numpy(), wl.dy[:n].cpu().numpy(),
                                            G.to_bits(wl.buf[:n * s.K]), s.act_dtype, n * s.K,
                                            row_base=a * s.K)
            assert (G.to_bits(wl.d_buf[:n * s.K]) == d_ref).all(), ("d_eo vs oracle", l, i)
            dx_ref = orc.dispatch_bwd(inv_h, d_ref, s.act_dtype, row_base=a * s.K)
            assert (wl.dx[:n].cpu().numpy().view(np.uint32) == dx_ref.view(np.uint32)).all(), ("dx vs oracle", l, i)
            err = np.abs(wl.dw[l, a:b].cpu().numpy().astype(np.float64) - dw_ref)
            scale = np.abs(dw_ref).max()
            assert err.max() <= 1e-4 * scale, ("dw vs oracle", l, i, float(err.max()), float(scale))


@pytest.mark.parametrize("cfg_id", [2, 3, 5])
def test_full_config_backward(cuda_device, cfg_id):
    cfg = synth.config(cfg_id)
    wl = bench.Workload(cfg, cuda_device, "update")
    wl.plan.plan()
    torch.cuda.synchronize()
    assert wl.plan.faults() == 0
    rng = np.random.default_rng(100 + cfg_id)
    inst = [wl.instances[k] for k in rng.choice(len(wl.instances), size=3, replace=False)]
    first, last = (0, 0), (cfg.L - 1, cfg.n_mb - 1)
    _backward_checks(wl, [first, last] + inst, {first, last})
    assert wl.plan.faults() == 0


@pytest.mark.parametrize("cfg_id,M", [(2, 2), (3, 8), (5, 4)])
def test_full_config_local(cuda_device, cfg_id, M):
    """Per-source, multi-machine Stage 4 at full size (bench.Workload with machines=M): invariants of
    the commodity plan for every instance, the locality rule and Eq.(5) traffic by torch library ops,
    O11 + O3/O4 on the first and last micro-step of layer 0, the data path on one instance."""
    cfg = synth.config(cfg_id)
    wl = bench.Workload(cfg, cuda_device, "recompute", M)
    lp, sv = wl.plan, wl.shape
    lp.plan()
    torch.cuda.synchronize()
    assert lp.faults() == 0 and sv.E == cfg.E * M
    _properties_all_instances(wl)                      # Eq.(8)/(9), offsets, bijection, stability on commodities
    R, S = cfg.P // M, cfg.S
    dev = lp.ids.device
    src_m = torch.from_numpy(wl.tok_src_h // R).to(dev).long()
    se = lp.real_slot_expert.long()                    # [L, S]
    mach_of_slot = (torch.arange(S, device=dev) // cfg.Ns) // R
    for l in range(cfg.L):
        ps = lp.pair_slot[l].long()                    # [T, K] = slot * M + source machine
        assert torch.equal(se[l][(ps // M).view(-1)], lp.real_ids[l].long().view(-1))
        assert torch.equal(ps % M, src_m[:, None].expand(-1, cfg.K))
        # locality: a pair leaves its machine only if that machine holds no copy of its expert
        holds = torch.zeros((cfg.E, M), dtype=torch.bool, device=dev)
        ok = se[l] >= 0
        holds[se[l][ok], mach_of_slot[ok]] = True
        crosses = mach_of_slot[ps // M] != src_m[:, None]
        assert not (crosses & holds[lp.real_ids[l].long(), src_m[:, None].expand(-1, cfg.K)]).any()
    q = lp.quota.long().view(cfg.n_mb, cfg.L, M, R * cfg.Ns, M)      # [.., machine of slot, slot in machine, source]
    assert torch.equal(lp.traffic.long(), q.sum(3).transpose(-1, -2))
    ids_h = lp.real_ids[0].cpu().numpy()
    for i in (0, cfg.n_mb - 1):
        a, b = int(wl.mb_off_h[i]), int(wl.mb_off_h[i + 1])
        key = np.repeat(wl.tok_src_h[a:b].astype(np.int64), cfg.K) * cfg.E + ids_h[a:b].reshape(-1)
        w_se = np.bincount(key, minlength=cfg.P * cfg.E).reshape(cfg.P, cfg.E).astype(np.int32)
        ref = orc.quota_local(w_se, wl.se_h[0], cfg.P, cfg.Ns, M)
        assert ref["fault"] == 0
        assert (lp.quota[i, 0].cpu().numpy() == ref["quota_v"]).all(), ("quota_v", i)
        assert (lp.rank_load[i, 0].cpu().numpy() == ref["rank_load"]).all()
        assert (lp.traffic[i, 0].cpu().numpy() == ref["traffic"]).all()
        se_v, f = orc.local_placement(wl.se_h[0], cfg.E, cfg.P, cfg.Ns, M)
        ids_v = (ids_h[a:b].astype(np.int64) * M + (wl.tok_src_h[a:b] // R)[:, None]).astype(np.int32)
        ps, inv, perm, f2 = orc.assign_instance(ids_v, se_v, ref["quota_v"], ref["slot_off_v"], cfg.E * M,
                                                base=a * cfg.K)
        assert f == 0 and f2 == 0
        assert (lp.pair_slot[0, a:b].cpu().numpy().ravel() == ps).all(), ("pair_slot_v", i)
        assert (lp.inv[0, a:b].cpu().numpy().ravel() == inv).all(), ("inv", i)
    _library_data_checks(wl, [wl.instances[0], wl.instances[-1]])


def test_full_config2_tradeoff(cuda_device):
    """Per-source Stage 4 under F = L_max + C_max at full size (bench.Workload with machines = 2,
    objective (1, 1)): invariants of the chosen commodity plan for every instance, F never above either
    end of the ladder, O15 on the first and last micro-step of layer 0, the data path on one instance."""
    cfg = synth.config(2)
    M = 2
    wl = bench.Workload(cfg, cuda_device, "recompute", M, "stage4", (1, 1))
    tp = wl.plan
    tp.plan()
    torch.cuda.synchronize()
    assert tp.faults() == 0
    # the plan's placement differs per instance: evaluate the invariants against the chosen one
    dev = tp.ids.device
    s = wl.shape
    quota, hist = tp.quota.long(), tp.hist.long()
    se = tp.slot_expert.long()                                        # [n_mb, L, S_v]
    per_e = torch.zeros((s.n_mb, s.L, s.E + 1), dtype=torch.int64, device=dev)
    per_e.scatter_add_(2, torch.where(se >= 0, se, torch.full_like(se, s.E)), quota)
    assert torch.equal(per_e[..., :s.E], hist) and (per_e[..., s.E] == 0).all()     # Eq.(8) / (9)
    assert torch.equal(tp.rank_load.long(), quota.view(s.n_mb, s.L, s.P, s.Ns).sum(-1))
    F = tp.F
    Fsel = F.gather(0, tp.member.long()[None]).squeeze(0)
    assert (Fsel == F.min(0).values).all() and (tp.member.long() == F.argmin(0)).all()
    R = cfg.P // M
    ids_h = tp.real_ids[0].cpu().numpy()
    for i in (0, cfg.n_mb - 1):
        a, b = int(wl.mb_off_h[i]), int(wl.mb_off_h[i + 1])
        key = np.repeat(wl.tok_src_h[a:b].astype(np.int64), cfg.K) * cfg.E + ids_h[a:b].reshape(-1)
        w_se = np.bincount(key, minlength=cfg.P * cfg.E).reshape(cfg.P, cfg.E).astype(np.int32)
        ref = orc.quota_tradeoff(w_se, wl.se_h[0], cfg.P, cfg.Ns, M, 1, 1)
        assert ref["fault"] == 0 and int(tp.member[i, 0]) == ref["member"]
        assert tp.F[:, i, 0].cpu().numpy().tolist() == ref["F"].tolist()
        assert (tp.quota[i, 0].cpu().numpy() == ref["quota_v"]).all()
        assert (tp.traffic[i, 0].cpu().numpy() == ref["traffic"]).all()
        ids_v = (ids_h[a:b].astype(np.int64) * M + (wl.tok_src_h[a:b] // R)[:, None]).astype(np.int32)
        ps, inv, perm, f = orc.assign_instance(ids_v, ref["se_v"], ref["quota_v"], ref["slot_off_v"], cfg.E * M,
                                               base=a * cfg.K)
        assert f == 0 and (tp.inv[0, a:b].cpu().numpy().ravel() == inv).all()
    _library_data_checks(wl, [wl.instances[0], wl.instances[-1]])
