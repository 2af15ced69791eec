"""GPU parity of the per-source, multi-machine Stage 4 (foremoe_source_ids, foremoe_local_placement,
foremoe_traffic + the unchanged hot path on the virtual shape) against the oracle O11 (and O1, O3/O4,
O5, O6 on the commodity instance), bit-exact."""
import dataclasses

import numpy as np
import pytest
import torch

from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import binding as fm
from paper_2606_11867_b200 import runner, synth
from tests import gpu_common as G

pytestmark = pytest.mark.gpu


def per_source_counts(ids_il, src_i, P, E):
    """w_{s,e} of one instance by numpy (library routine): [P, E]."""
    K = ids_il.shape[1]
    key = np.repeat(src_i.astype(np.int64), K) * E + ids_il.reshape(-1)
    return np.bincount(key, minlength=P * E).reshape(P, E).astype(np.int32)


def local_plan(shape, M, ids, w, mb_off, se, tok_src):
    t = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).to(G.DEV)
    lp = runner.LocalStepPlan(shape, M, t(ids, torch.int32), t(w, torch.float32), t(mb_off, torch.int32),
                              t(se, torch.int32), t(tok_src, torch.int32))
    for name in ("ids", "slot_expert", "hist", "quota", "rank_load", "slot_off", "pair_slot", "inv", "traffic"):
        getattr(lp, name).fill_(-77)
    lp.plan()
    torch.cuda.synchronize()
    return lp


def check_local(cfg, M, layers=None, data_instances=(), what=""):
    ids, w, mb_off, se = G.make_case(cfg)
    tok_src = synth.gen_tok_src(cfg)
    shape = fm.shape_of(cfg)
    R = cfg.P // M
    lp = local_plan(shape, M, ids, w, mb_off, se, tok_src)
    assert lp.faults() == 0
    sv = lp.shape
    assert (sv.E, sv.Nb, sv.Nr, sv.S) == (cfg.E * M, cfg.Nb * M, cfg.Nr * M, cfg.S * M)
    # the virtual instance
    ids_v = ids.astype(np.int64) * M + (tok_src // R)[None, :, None]
    assert (lp.ids.cpu().numpy() == ids_v).all(), (what, "ids_v")
    se_v_g = lp.slot_expert.cpu().numpy()
    hist_v = lp.hist.cpu().numpy()
    layers = range(cfg.L) if layers is None else layers
    for l in layers:
        ref_se_v, f = orc.local_placement(se[l], cfg.E, cfg.P, cfg.Ns, M)
        assert f == 0 and (se_v_g[l] == ref_se_v).all(), (what, "slot_expert_v", l)
        for i in range(cfg.n_mb):
            a, b = int(mb_off[i]), int(mb_off[i + 1])
            w_se = per_source_counts(ids[l, a:b], tok_src[a:b], cfg.P, cfg.E)
            # hist_v[e*M + m] = w_{s,e} summed over the sources of machine m
            agg = w_se.reshape(M, R, cfg.E).sum(1)                   # [M, E]
            assert (hist_v[i, l].reshape(cfg.E, M) == agg.T).all(), (what, "hist_v", l, i)
            ref = orc.quota_local(w_se, se[l], cfg.P, cfg.Ns, M)
            assert ref["fault"] == 0
            assert (lp.quota[i, l].cpu().numpy() == ref["quota_v"]).all(), (what, "quota_v", l, i)
            assert (lp.rank_load[i, l].cpu().numpy() == ref["rank_load"]).all(), (what, "rank_load", l, i)
            assert (lp.slot_off[i, l].cpu().numpy() == ref["slot_off_v"]).all(), (what, "slot_off_v", l, i)
            assert (lp.traffic[i, l].cpu().numpy() == ref["traffic"]).all(), (what, "traffic", l, i)
            ps, inv, perm, f = orc.assign_instance(ids_v[l, a:b].astype(np.int32), ref_se_v, ref["quota_v"],
                                                   ref["slot_off_v"], cfg.E * M, base=a * cfg.K)
            assert f == 0
            assert (lp.pair_slot[l, a:b].cpu().numpy().ravel() == ps).all(), (what, "pair_slot_v", l, i)
            assert (lp.inv[l, a:b].cpu().numpy().ravel() == inv).all(), (what, "inv", l, i)
            # every pair sits on a slot that really holds its expert, from its own source machine
            assert (se[l][ps // M] == ids[l, a:b].ravel()).all()
            assert ((ps % M) == np.repeat(tok_src[a:b] // R, cfg.K)).all()
            if (l, i) in data_instances and b > a:
                n = b - a
                x = synth.gen_activations(cfg, n, i, G.DEV)
                perm_g = torch.full((n * cfg.K,), -5, dtype=torch.int32, device=G.DEV)
                buf = torch.empty((n * cfg.K, cfg.H), dtype=shape.act_torch_dtype, device=G.DEV)
                y = torch.empty((n, cfg.H), dtype=torch.float32, device=G.DEV)
                lp.dispatch(l, i, i + 1, x, perm_g, buf)
                lp.combine(l, i, i + 1, buf, y)
                torch.cuda.synchronize()
                assert (perm_g.cpu().numpy() == perm).all(), (what, "perm", l, i)
                buf_ref = orc.gather(perm, G.to_bits(x), cfg.K, pair_base=a * cfg.K)
                assert (G.to_bits(buf) == buf_ref).all(), (what, "buf", l, i)
                y_ref = orc.combine(inv.reshape(n, cfg.K), w[l, a:b], buf_ref, cfg.act_dtype, row_base=a * cfg.K)
                assert (y.cpu().numpy().view(np.uint32) == y_ref.view(np.uint32)).all(), (what, "y", l, i)
    return lp


@pytest.mark.parametrize("M", [1, 2, 4])
def test_tiny_config1_local(cuda_device, M):
    cfg = synth.config(1)
    check_local(cfg, M, data_instances={(0, 0), (0, cfg.n_mb - 1)}, what=f"cfg1-M{M}")


@pytest.mark.parametrize("cfg_id,kw,M", [
    (2, dict(L=2, n_samples=12, sample_len=700, H=256, mb_samples=4), 2),
    (2, dict(L=1, n_samples=8, sample_len=500, H=128, mb_samples=4), 8),     # M = P: w_{s,e} itself
    (3, dict(L=1, n_samples=4, sample_len=1100, H=256, mb_samples=2), 8),
    (5, dict(L=1, n_samples=2, sample_len=3000, H=256, mb_samples=1), 4),
    (4, dict(L=1, n_samples=9, H=128, mb_samples=2), 2),
])
def test_scaled_configs_local(cuda_device, cfg_id, kw, M):
    cfg = synth.config(cfg_id).scaled(**kw)
    lp = check_local(cfg, M, data_instances={(0, 0)}, what=f"cfg{cfg_id}-M{M}")
    tr = lp.traffic.cpu().numpy().astype(np.int64)
    assert (tr.sum((-1, -2)) == lp.rank_load.cpu().numpy().sum(-1)).all()


def test_locality_effect(cuda_device):
    """With replicas spread over machines the localized plan moves fewer tokens across machines than
    the plain Stage 4 (whose choice ignores the source), at an equal or higher max rank load."""
    cfg = synth.config(2).scaled(L=2, n_samples=16, sample_len=600, H=128, mb_samples=4)
    M, R = 2, cfg.P // 2
    ids, w, mb_off, se = G.make_case(cfg)
    tok_src = synth.gen_tok_src(cfg)
    lp = local_plan(fm.shape_of(cfg), M, ids, w, mb_off, se, tok_src)
    sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se)
    tr = lp.traffic.cpu().numpy().astype(np.int64)
    cross_local = tr.sum((-1, -2)) - np.trace(tr, axis1=-2, axis2=-1)
    ps = sp.pair_slot.cpu().numpy()
    for l in range(cfg.L):
        for i in range(cfg.n_mb):
            a, b = int(mb_off[i]), int(mb_off[i + 1])
            dst_m = (ps[l, a:b] // cfg.Ns) // R
            src_m = (tok_src[a:b] // R)[:, None]
            cross_plain = int((dst_m != src_m).sum())
            assert cross_local[i, l] <= cross_plain
            assert lp.rank_load[i, l].max().item() >= sp.rank_load[i, l].max().item()


def test_local_faults_and_errors(cuda_device):
    cfg = synth.config(1)
    ids, w, mb_off, se = G.make_case(cfg)
    shape = fm.shape_of(cfg)
    tok_src = synth.gen_tok_src(cfg)
    bad = tok_src.copy()
    bad[5] = cfg.P
    lp = local_plan(shape, 2, ids, w, mb_off, se, bad)
    assert lp.faults() & fm.FAULT_SOURCE
    assert (lp.ids[0, 5].cpu().numpy() == -1).all()
    se_bad = se.copy()
    se_bad[0, 1] = cfg.E
    lp = local_plan(shape, 2, ids, w, mb_off, se_bad, tok_src)
    assert lp.faults() & fm.FAULT_SLOT_EXPERT
    t = lambda a: torch.as_tensor(a, dtype=torch.int32).to(G.DEV)
    with pytest.raises(fm.ForeMoEError):
        fm.source_ids(shape, 3, t(ids), t(tok_src), torch.empty_like(t(ids)))       # 3 does not divide P = 4
    with pytest.raises(fm.ForeMoEError):
        fm.traffic(shape, 0, t(ids), t(ids))
