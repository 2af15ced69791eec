"""GPU parity of foremoe_base_placement / foremoe_microstep_placement against the oracle (O7 / O8),
bit-exact, and the end-to-end effect: Stage 4 on the per-micro-step placements."""
import dataclasses

import numpy as np
import pytest
import torch

from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import binding as fm
from paper_2606_11867_b200 import synth
from tests import gpu_common as G

pytestmark = pytest.mark.gpu


def _gpu_placements(shape, hist, step, M):
    dev = G.DEV
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    base = torch.full((shape.L, shape.S), -7, dtype=torch.int32, device=dev)
    fm.base_placement(shape, torch.as_tensor(step, dtype=torch.int64).to(dev), base, st)
    mb = torch.full((shape.n_mb, shape.L, shape.S), -7, dtype=torch.int32, device=dev)
    fm.microstep_placement(shape, M, torch.as_tensor(hist, dtype=torch.int32).to(dev), base, mb, st)
    torch.cuda.synchronize()
    return base.cpu().numpy(), mb.cpu().numpy(), int(st.item())


@pytest.mark.parametrize("seed", range(6))
def test_random_instances(cuda_device, seed):
    rng = np.random.default_rng(50 + seed)
    P = [2, 4, 6, 8, 64, 40][seed]
    Nb, Nr = [3, 2, 4, 16, 4, 1][seed], [1, 2, 0, 2, 1, 3][seed]
    M = [1, 2, 3, 1, 8, 1][seed]
    E, L, n_mb = P * Nb, 5, 6
    shape = fm.Shape(L=L, E=E, K=1, P=P, Nb=Nb, Nr=Nr, T=8, n_mb=n_mb, H=8, act_dtype=fm.ACT_FP32)
    hist = (rng.integers(0, 500, size=(n_mb, L, E)) * rng.integers(0, 2, size=(n_mb, L, E))).astype(np.int32)
    hist[1] = 7                                   # all-equal loads: pure tie-breaking
    hist[2] = 0                                   # empty micro-step: nothing is replicated
    step = hist.astype(np.int64).sum(0)
    base, mb, fault = _gpu_placements(shape, hist, step, M)
    assert fault == 0
    for l in range(L):
        ref, f = orc.base_placement(step[l], P, Nb, Nr)
        assert f == 0 and (base[l] == ref).all(), ("base", l)
        for i in range(n_mb):
            ref2, f = orc.microstep_placement(hist[i, l], ref, P, Nb, Nr, M)
            assert f == 0 and (mb[i, l] == ref2).all(), ("microstep", i, l)


def test_golden_vector_on_gpu(cuda_device):
    c = np.array([10, 9, 8, 7, 3, 2, 1, 1])
    shape = fm.Shape(L=1, E=8, K=1, P=4, Nb=2, Nr=1, T=8, n_mb=1, H=8, act_dtype=fm.ACT_FP32)
    base, mb, fault = _gpu_placements(shape, c.reshape(1, 1, 8).astype(np.int32), c.reshape(1, 8), 1)
    assert fault == 0
    assert base.reshape(4, 3).tolist() == [[0, 7, -1], [1, 6, -1], [2, 5, -1], [3, 4, -1]]
    assert mb.reshape(4, 3).tolist() == [[0, 7, 1], [1, 6, 0], [2, 5, 3], [3, 4, 2]]


def test_faults(cuda_device):
    shape = fm.Shape(L=1, E=4, K=1, P=2, Nb=2, Nr=1, T=8, n_mb=2, H=8, act_dtype=fm.ACT_FP32)
    hist = np.array([[[3, 2, 1, 1]], [[3, -2, 1, 1]]], dtype=np.int32)
    dev = G.DEV
    base = torch.tensor([[0, 3, -1, 1, 2, -1]], dtype=torch.int32, device=dev)
    out = torch.full((2, 1, 6), -7, dtype=torch.int32, device=dev)
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    fm.microstep_placement(shape, 1, torch.from_numpy(hist).to(dev), base, out, st)
    assert int(st.item()) == fm.FAULT_ID_RANGE
    assert (out[1].cpu().numpy() == -1).all() and (out[0].cpu().numpy() >= -1).all()
    st.zero_()
    bad = base.clone(); bad[0, 1] = -1                      # expert 3 has no base slot
    fm.microstep_placement(shape, 1, torch.from_numpy(hist).to(dev), bad, out, st)
    assert int(st.item()) & fm.FAULT_SLOT_EXPERT
    with pytest.raises(fm.ForeMoEError):
        fm.microstep_placement(shape, 3, torch.from_numpy(hist).to(dev), base, out, st)   # P % M != 0


@pytest.mark.parametrize("cfg_id,kw", [(3, dict(L=2, n_samples=16, sample_len=1500, H=256)),
                                       (2, dict(L=2, n_samples=16, sample_len=800, H=256, mb_samples=4))])
def test_stages_2_to_4_pipeline(cuda_device, cfg_id, kw):
    """hist -> base placement -> per-micro-step placements -> assign (placement_mb_stride) ->
    dispatch / combine: every array equals the oracle chain, and max rank load is no worse than with
    the step-level placement on every instance."""
    cfg = synth.config(cfg_id).scaled(**kw)
    ids, w, mb_off = synth.gen_trace(cfg, "cpu")
    ids, w, mb_off = ids.numpy(), w.numpy(), mb_off.numpy()
    hist, step, f = orc.load_hist(ids, mb_off, cfg.E)
    s0 = fm.shape_of(cfg)
    base, mb, fault = _gpu_placements(s0, hist, step, 1)
    assert fault == 0
    shape = dataclasses.replace(s0, placement_mb_stride=s0.L * s0.S)
    sp = G.gpu_plan(shape, ids, w, mb_off, mb)
    assert sp.faults() == 0
    step_level = synth.gen_placement(cfg, step)
    K = cfg.K
    for l in range(cfg.L):
        b_ref, f = orc.base_placement(step[l], cfg.P, cfg.Nb, cfg.Nr)
        assert (base[l] == b_ref).all()
        for i in range(cfg.n_mb):
            a, b = int(mb_off[i]), int(mb_off[i + 1])
            se, f = orc.microstep_placement(hist[i, l], b_ref, cfg.P, cfg.Nb, cfg.Nr, 1)
            assert f == 0 and (mb[i, l] == se).all()
            q, rl, so, _, f = orc.quota(hist[i, l], se, cfg.P, cfg.Ns)
            ps, inv, perm, f2 = orc.assign_instance(ids[l, a:b], se, q, so, cfg.E, base=a * K)
            assert f == 0 and f2 == 0
            assert (sp.quota[i, l].cpu().numpy() == q).all()
            assert (sp.rank_load[i, l].cpu().numpy() == rl).all()
            assert (sp.inv[l, a:b].cpu().numpy().ravel() == inv).all()
            _, rl0, _, _, _ = orc.quota(hist[i, l], step_level[l], cfg.P, cfg.Ns)
            assert rl.max() <= rl0.max()
    # data path on the per-micro-step plan
    ref = dict(perm=np.zeros((cfg.L, cfg.T * K), dtype=np.int32), inv=sp.inv.cpu().numpy())
    for l in range(cfg.L):
        for i in range(cfg.n_mb):
            a, b = int(mb_off[i]) * K, int(mb_off[i + 1]) * K
            ref["perm"][l, ref["inv"][l].ravel()[a:b]] = np.arange(a, b)
    x = G.activations(cfg, mb_off, range(cfg.n_mb))
    G.check_data_path(sp, ref, x, range(cfg.L), range(cfg.n_mb), "stages2-4")


# ------------------------------------------------------------------ Alg. 2 Stage 2 (swap relocation, O12)
def _swap_gpu(shape, M, win, rounds, a, b, hist_v, base):
    dev = G.DEV
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    out = torch.full((shape.n_mb, shape.L, shape.S), -7, dtype=torch.int32, device=dev)
    nr = torch.full((shape.n_mb, shape.L), -7, dtype=torch.int32, device=dev)
    fm.swap_relocation(shape, M, win, rounds, a, b, torch.as_tensor(hist_v, dtype=torch.int32).to(dev),
                       torch.as_tensor(base, dtype=torch.int32).to(dev), out, nr, st)
    torch.cuda.synchronize()
    return out.cpu().numpy(), nr.cpu().numpy(), int(st.item())


@pytest.mark.parametrize("seed", range(8))
def test_swap_relocation_random(cuda_device, seed):
    rng = np.random.default_rng(70 + seed)
    P, M, Nb, Nr = [(2, 1, 2, 1), (4, 2, 4, 1), (8, 2, 16, 2), (8, 8, 4, 0), (64, 8, 4, 1), (32, 4, 16, 4),
                    (6, 3, 5, 2), (40, 1, 3, 1)][seed]
    win = [2, 1, 4, 3, 2, 40, 2, 3][seed]
    a, b = [(1, 0), (1, 1), (3, 2), (0, 1), (1, 1), (2, 1), (1, 5), (1, 0)][seed]
    E, L, n_mb, Ns = P * Nb, 3, 5, Nb + Nr
    shape = fm.Shape(L=L, E=E, K=1, P=P, Nb=Nb, Nr=Nr, T=8, n_mb=n_mb, H=8, act_dtype=fm.ACT_FP32)
    hist_v = (rng.integers(0, 400, size=(n_mb, L, E, M)) * (rng.random((n_mb, L, E, M)) < 0.8)).astype(np.int32)
    hist_v[1] = 9                                     # all equal: nothing to gain, pure tie handling
    hist_v[2, :, : E // 2] = 0                        # many zero loads
    base = np.full((L, P * Ns), -1, dtype=np.int32)
    for l in range(L):
        perm = rng.permutation(E)
        for r in range(P):
            base[l, r * Ns:r * Ns + Nb] = perm[r * Nb:(r + 1) * Nb]
            base[l, r * Ns + Nb:(r + 1) * Ns] = -1
    out, nr, fault = _swap_gpu(shape, M, win, 24, a, b, hist_v.reshape(n_mb, L, E * M), base)
    assert fault == 0
    moved = 0
    for i in range(n_mb):
        for l in range(L):
            ref, st, f = orc.swap_relocation(hist_v[i, l].T.copy(), base[l], P, Nb, Nr, M, win, 24, a, b)
            assert f == 0 and (out[i, l] == ref).all(), ("swap", i, l)
            assert nr[i, l] == st[0]
            moved += int(st[0])
    assert moved > 0
    # fewer rounds allowed: the prefix of the same sequence
    out2, nr2, _ = _swap_gpu(shape, M, win, 1, a, b, hist_v.reshape(n_mb, L, E * M), base)
    ref, st, f = orc.swap_relocation(hist_v[0, 0].T.copy(), base[0], P, Nb, Nr, M, win, 1, a, b)
    assert (out2[0, 0] == ref).all() and nr2[0, 0] == st[0]


def test_swap_relocation_golden_and_faults(cuda_device):
    shape = fm.Shape(L=1, E=4, K=1, P=2, Nb=2, Nr=1, T=8, n_mb=1, H=8, act_dtype=fm.ACT_FP32)
    base = np.array([[0, 1, -1, 2, 3, -1]], dtype=np.int32)
    out, nr, fault = _swap_gpu(shape, 1, 2, 8, 1, 0, np.array([[[9, 8, 1, 2]]]), base)
    assert fault == 0 and out.reshape(2, 3).tolist() == [[3, 1, -1], [2, 0, -1]] and nr.item() == 1
    hv = np.array([[5, 0, 6, 1], [1, 2, 0, 7]]).T.reshape(1, 1, 8)            # [e*M + m]
    out, nr, fault = _swap_gpu(shape, 2, 2, 8, 0, 1, hv, base)
    assert fault == 0 and out.reshape(2, 3).tolist() == [[0, 2, -1], [1, 3, -1]] and nr.item() == 1
    bad = base.copy(); bad[0, 1] = 0
    out, nr, fault = _swap_gpu(shape, 1, 2, 8, 1, 0, np.array([[[9, 8, 1, 2]]]), bad)
    assert fault & fm.FAULT_SLOT_EXPERT and (out == -1).all()
    out, nr, fault = _swap_gpu(shape, 1, 2, 8, 1, 0, np.array([[[9, -8, 1, 2]]]), base)
    assert fault & fm.FAULT_ID_RANGE and (out == -1).all()
    with pytest.raises(fm.ForeMoEError):
        _swap_gpu(shape, 3, 2, 8, 1, 0, np.zeros((1, 1, 12)), base)           # 3 does not divide P
    with pytest.raises(fm.ForeMoEError):
        _swap_gpu(shape, 1, 0, 8, 1, 0, np.zeros((1, 1, 4)), base)            # empty window


def test_swap_then_stage4_on_config_trace(cuda_device):
    """End to end on a config-2-shaped trace: load_hist -> base placement -> swap relocation ->
    foremoe_assign on the per-micro-step placements; the max rank load never gets worse than with
    the base placement alone, and the plan stays consistent with the oracle."""
    cfg = synth.config(2).scaled(L=2, n_samples=16, sample_len=512, H=64, mb_samples=4)
    ids, w, mb_off, _ = G.make_case(cfg)
    shape = fm.shape_of(cfg)
    hist, step, _ = orc.load_hist(ids, mb_off, cfg.E)
    base = np.stack([orc.base_placement(step[l], cfg.P, cfg.Nb, cfg.Nr)[0] for l in range(cfg.L)])
    out, nr, fault = _swap_gpu(shape, 1, 4, 32, 1, 0, hist, base)
    assert fault == 0
    sp0 = G.gpu_plan(shape, ids, w, mb_off, base)
    shape_mb = dataclasses.replace(shape, placement_mb_stride=shape.L * shape.S)
    sp1 = G.gpu_plan(shape_mb, ids, w, mb_off, out)
    assert sp0.faults() == 0 and sp1.faults() == 0
    m0 = sp0.rank_load.max(-1).values.cpu().numpy()
    m1 = sp1.rank_load.max(-1).values.cpu().numpy()
    assert (m1 <= m0).all() and (m1 < m0).any()
    for i in range(cfg.n_mb):
        for l in range(cfg.L):
            q, rl, so, _, f = orc.quota(hist[i, l], out[i, l], cfg.P, cfg.Ns)
            assert f == 0 and (sp1.quota[i, l].cpu().numpy() == q).all()


# ------------------------------------------------------------------ Stage 3 alone (O13) after the swaps
@pytest.mark.parametrize("seed", range(5))
def test_replication_after_swaps(cuda_device, seed):
    rng = np.random.default_rng(90 + seed)
    P, M, Nb, Nr = [(4, 1, 4, 1), (8, 2, 16, 2), (64, 8, 4, 1), (32, 1, 16, 4), (6, 3, 5, 2)][seed]
    E, L, n_mb, Ns = P * Nb, 2, 4, Nb + Nr
    shape = fm.Shape(L=L, E=E, K=1, P=P, Nb=Nb, Nr=Nr, T=8, n_mb=n_mb, H=8, act_dtype=fm.ACT_FP32)
    hist = (rng.integers(0, 400, size=(n_mb, L, E)) * (rng.random((n_mb, L, E)) < 0.8)).astype(np.int32)
    hist[3] = 0
    base = np.full((L, P * Ns), -1, dtype=np.int32)
    for l in range(L):
        perm = rng.permutation(E)
        for r in range(P):
            base[l, r * Ns:r * Ns + Nb] = perm[r * Nb:(r + 1) * Nb]
    swapped, nr, fault = _swap_gpu(shape, 1, 3, 16, 1, 0, hist, base)
    assert fault == 0
    dev = G.DEV
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    buf = torch.as_tensor(swapped).to(dev)
    buf.view(n_mb, L, P, Ns)[..., Nb:] = -9                     # redundant slots of the input are not read
    fm.replication(shape, M, torch.as_tensor(hist).to(dev), buf, buf, st)        # in place
    torch.cuda.synchronize()
    got = buf.cpu().numpy()
    assert int(st.item()) == 0
    for i in range(n_mb):
        for l in range(L):
            ref, f = orc.replication(hist[i, l], swapped[i, l], P, Nb, Nr, M)
            assert f == 0 and (got[i, l] == ref).all(), ("replication", i, l)
    # fault: an expert twice in the base slots of one instance -> that instance is all -1, others fine
    bad = torch.as_tensor(swapped).to(dev)
    bad[1, 0, 0] = bad[1, 0, 1]
    out = torch.empty_like(bad)
    fm.replication(shape, M, torch.as_tensor(hist).to(dev), bad, out, st)
    torch.cuda.synchronize()
    assert int(st.item()) & fm.FAULT_SLOT_EXPERT
    assert (out[1, 0] == -1).all() and (out[0, 0].cpu().numpy() == got[0, 0]).all()


# ------------------------------------------------------------------ Alg. 1 in full (O14)
@pytest.mark.parametrize("seed", range(6))
def test_base_placement_machines(cuda_device, seed):
    rng = np.random.default_rng(120 + seed)
    P, M, Nb, Nr = [(4, 2, 2, 1), (8, 2, 16, 2), (64, 8, 4, 1), (32, 4, 16, 4), (6, 3, 5, 0), (64, 64, 4, 1)][seed]
    a, b = [(1, 1), (1, 0), (3, 2), (0, 1), (1, 5), (2, 1)][seed]
    E, L = P * Nb, 4
    shape = fm.Shape(L=L, E=E, K=1, P=P, Nb=Nb, Nr=Nr, T=8, n_mb=1, H=8, act_dtype=fm.ACT_FP32)
    tot = (rng.integers(0, 5000, size=(L, E, M)) * (rng.random((L, E, M)) < 0.7)).astype(np.int64)
    tot[1] = 11                                       # all equal: ties only
    tot[2, :, 1:] = 0                                 # every token from machine 0
    dev = G.DEV
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    out = torch.full((L, shape.S), -7, dtype=torch.int32, device=dev)
    fm.base_placement_machines(shape, M, a, b, torch.as_tensor(tot.reshape(L, E * M)).to(dev), out, st)
    torch.cuda.synchronize()
    assert int(st.item()) == 0
    got = out.cpu().numpy()
    for l in range(L):
        ref, f = orc.base_placement_machines(tot[l].T.copy(), P, Nb, Nr, M, a, b)
        assert f == 0 and (got[l] == ref).all(), ("alg1", l)
    # M = 1 through the same entry equals foremoe_base_placement
    out1 = torch.empty_like(out)
    out7 = torch.empty_like(out)
    step = torch.as_tensor(tot.sum(-1)).to(dev)
    fm.base_placement_machines(shape, 1, 1, 0, step, out1, st)
    fm.base_placement(shape, step, out7, st)
    torch.cuda.synchronize()
    assert torch.equal(out1, out7)
    neg = tot.reshape(L, E * M).copy(); neg[3, 5] = -2
    fm.base_placement_machines(shape, M, a, b, torch.as_tensor(neg).to(dev), out, st)
    torch.cuda.synchronize()
    assert int(st.item()) & fm.FAULT_ID_RANGE and (out[3] == -1).all() and (out[0].cpu().numpy() == got[0]).all()
    with pytest.raises(fm.ForeMoEError):
        fm.base_placement_machines(shape, M, -1, b, torch.as_tensor(neg).to(dev), out, st)


# ------------------------------------------------------------------ Alg. 2 Stage 3: replica search (O16)
@pytest.mark.parametrize("seed", range(8))
def test_replica_search(cuda_device, seed):
    """foremoe_replica_search against oracle O16 on random instances: placements bit for bit, number of
    replicas and objective before / after; the golden four-round vector; faults."""
    rng = np.random.default_rng(600 + seed)
    P, M, Nb, Nr = [(4, 1, 2, 1), (4, 2, 1, 1), (8, 2, 4, 2), (8, 4, 2, 2), (6, 3, 3, 1), (16, 4, 4, 1),
                    (8, 8, 2, 2), (32, 8, 2, 1)][seed]
    a, b = [(1, 0), (1, 1), (2, 1), (1, 3), (1, 1), (3, 2), (1, 2), (1, 1)][seed]
    maxc = [8, 8, 3, 2, 8, 4, 8, 8][seed]
    E, L, n_mb, Ns = P * Nb, 2, 5, Nb + Nr
    shape = fm.Shape(L=L, E=E, K=1, P=P, Nb=Nb, Nr=Nr, T=8, n_mb=n_mb, H=8, act_dtype=fm.ACT_FP32)
    hv = (rng.integers(0, 80, size=(n_mb, L, E, M)) * (rng.random((n_mb, L, E, M)) < 0.7)).astype(np.int32)
    hot = rng.choice(E, size=max(1, E // 6), replace=False)
    hv[:, :, hot] *= 7
    hv[4] = 0                                                         # an empty micro-step: nothing to place
    hv[3, 1] = 5                                                      # all equal: ties only
    placed = np.full((n_mb, L, P, Ns), -1, dtype=np.int32)
    for i in range(n_mb):
        for l in range(L):
            placed[i, l, :, :Nb] = rng.permutation(E).reshape(P, Nb)
    placed[..., Nb:] = rng.integers(-1, E, size=(n_mb, L, P, Nr))     # garbage: not read
    dev = G.DEV
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    t = lambda x, dt=torch.int32: torch.as_tensor(np.ascontiguousarray(x), dtype=dt).to(dev)
    out = torch.full((n_mb, L, P * Ns), -7, dtype=torch.int32, device=dev)
    reps = torch.full((n_mb, L), -7, dtype=torch.int32, device=dev)
    F = torch.full((n_mb, L, 2), -7, dtype=torch.int64, device=dev)
    fm.replica_search(shape, M, maxc, a, b, t(hv.reshape(n_mb, L, E * M)), t(placed.reshape(n_mb, L, -1)), out, reps, F, st)
    torch.cuda.synchronize()
    assert int(st.item()) == 0
    got, nrep, Fg = out.cpu().numpy(), reps.cpu().numpy(), F.cpu().numpy()
    total = 0
    for i in range(n_mb):
        for l in range(L):
            ref, stats, f = orc.replica_search(hv[i, l].T.copy(), placed[i, l].ravel(), P, Nb, Nr, M, a, b, max_copies=maxc)
            assert f == 0
            assert (got[i, l] == ref).all(), ("replica_search", seed, i, l, got[i, l].tolist(), ref.tolist())
            assert nrep[i, l] == stats[0] and Fg[i, l].tolist() == [int(stats[1]), int(stats[2])]
            total += int(stats[0])
    assert total > 0 and nrep[4].sum() == 0
    # in place, and without the optional outputs
    buf = t(placed.reshape(n_mb, L, -1))
    fm.replica_search(shape, M, maxc, a, b, t(hv.reshape(n_mb, L, E * M)), buf, buf, None, None, st)
    torch.cuda.synchronize()
    assert torch.equal(buf, out)


@pytest.mark.parametrize("P,M,Nb", [(4, 2, 2), (8, 1, 4), (6, 3, 1)])
def test_replica_search_without_redundant_slots(cuda_device, P, M, Nb):
    """N_r = 0: there is nothing to place, no round runs, and the objective "before" is still the true
    objective of the base placement (equal to "after"), as in O16 which evaluates it ahead of the loop."""
    rng = np.random.default_rng(P * 100 + M)
    E, L, n_mb, a, b = P * Nb, 2, 3, 2, 3
    shape = fm.Shape(L=L, E=E, K=1, P=P, Nb=Nb, Nr=0, T=8, n_mb=n_mb, H=8, act_dtype=fm.ACT_FP32)
    hv = rng.integers(1, 80, size=(n_mb, L, E, M)).astype(np.int32)
    placed = np.stack([rng.permutation(E) for _ in range(n_mb * L)]).reshape(n_mb, L, E).astype(np.int32)
    dev = G.DEV
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    t = lambda x, dt=torch.int32: torch.as_tensor(np.ascontiguousarray(x), dtype=dt).to(dev)
    out = torch.full((n_mb, L, E), -7, dtype=torch.int32, device=dev)
    reps = torch.full((n_mb, L), -7, dtype=torch.int32, device=dev)
    F = torch.full((n_mb, L, 2), -7, dtype=torch.int64, device=dev)
    fm.replica_search(shape, M, 8, a, b, t(hv.reshape(n_mb, L, E * M)), t(placed), out, reps, F, st)
    torch.cuda.synchronize()
    assert int(st.item()) == 0 and (reps == 0).all()
    Fg = F.cpu().numpy()
    for i in range(n_mb):
        for l in range(L):
            ref, stats, f = orc.replica_search(hv[i, l].T.copy(), placed[i, l], P, Nb, 0, M, a, b, max_copies=8)
            assert f == 0 and stats[0] == 0 and stats[1] == stats[2] > 0
            assert (out[i, l].cpu().numpy() == ref).all()
            assert Fg[i, l].tolist() == [int(stats[1]), int(stats[2])], (i, l, Fg[i, l].tolist(), stats)


def test_replica_search_golden_faults_and_pipeline(cuda_device):
    import json, os
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "replica_search_vectors.json")))["vectors"][0]
    P, Nb, Nr, M = g["P"], g["Nb"], g["Nr"], g["M"]
    E = P * Nb
    shape = fm.Shape(L=1, E=E, K=1, P=P, Nb=Nb, Nr=Nr, T=8, n_mb=1, H=8, act_dtype=fm.ACT_FP32)
    dev = G.DEV
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    t = lambda x, dt=torch.int32: torch.as_tensor(np.ascontiguousarray(x), dtype=dt).to(dev)
    hv = np.array(g["c_me"], dtype=np.int32).T.reshape(1, 1, E * M)             # [e*M + m]
    out = torch.empty((1, 1, P * (Nb + Nr)), dtype=torch.int32, device=dev)
    reps = torch.empty((1, 1), dtype=torch.int32, device=dev)
    F = torch.empty((1, 1, 2), dtype=torch.int64, device=dev)
    fm.replica_search(shape, M, g["max_copies"], g["a"], g["b"], t(hv), t(np.array(g["placed"]).reshape(1, 1, -1)), out, reps, F, st)
    torch.cuda.synchronize()
    assert out.view(P, -1).tolist() == g["out"] and [int(reps.item())] + F.view(-1).tolist() == g["stats"]
    # faults: an expert twice in the base slots; a negative load
    bad = np.array(g["placed"]).reshape(1, 1, -1).copy(); bad[0, 0, 0] = bad[0, 0, 2]
    fm.replica_search(shape, M, 8, 1, 1, t(hv), t(bad), out, reps, F, st)
    torch.cuda.synchronize()
    assert int(st.item()) & fm.FAULT_SLOT_EXPERT and (out == -1).all()
    with pytest.raises(fm.ForeMoEError):
        fm.replica_search(shape, 3, 8, 1, 1, t(hv), t(bad), out, reps, F, st)          # 3 does not divide P
    with pytest.raises(fm.ForeMoEError):
        fm.replica_search(shape, M, 40, 1, 1, t(hv), t(bad), out, reps, F, st)         # max_copies > 31
    # Alg. 2 end to end on a config-2-shaped trace: Stage 1 -> swaps -> replica search -> Stage 4
    cfg = synth.config(2).scaled(L=2, n_samples=16, sample_len=512, H=64, mb_samples=4)
    ids, w, mb_off, _ = G.make_case(cfg)
    shape = fm.shape_of(cfg)
    hist, step, _ = orc.load_hist(ids, mb_off, cfg.E)
    base = np.stack([orc.base_placement(step[l], cfg.P, cfg.Nb, cfg.Nr)[0] for l in range(cfg.L)])
    swapped, nr, fault = _swap_gpu(shape, 1, 4, 32, 1, 0, hist, base)
    assert fault == 0
    st.zero_()
    full = torch.empty((cfg.n_mb, cfg.L, cfg.S), dtype=torch.int32, device=dev)
    fm.replica_search(shape, 1, 8, 1, 0, t(hist), t(swapped), full, None, None, st)
    torch.cuda.synchronize()
    assert int(st.item()) == 0
    for i in range(cfg.n_mb):
        for l in range(cfg.L):
            ref, _, f = orc.replica_search(hist[i, l], swapped[i, l], cfg.P, cfg.Nb, cfg.Nr, 1, 1, 0)
            assert f == 0 and (full[i, l].cpu().numpy() == ref).all()
    shape_mb = dataclasses.replace(shape, placement_mb_stride=shape.L * shape.S)
    sp_sw = G.gpu_plan(shape_mb, ids, w, mb_off, swapped)
    sp_rs = G.gpu_plan(shape_mb, ids, w, mb_off, full.cpu().numpy())
    assert sp_sw.faults() == 0 and sp_rs.faults() == 0
    m_sw = sp_sw.rank_load.max(-1).values
    m_rs = sp_rs.rank_load.max(-1).values
    assert (m_rs <= m_sw).all() and (m_rs < m_sw).any()                # replicas + Stage 4 only help
