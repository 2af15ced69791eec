"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by
element, on the same seeded inputs.  Bit-exact for every integer output and gathered row; the
fp32 combine within max relative error 1e-6 (BASELINE.json north_star) -- and, since both sides
use the same fma order (reading 16), bit-identical.
"""
import numpy as np
import pytest
import torch

from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import binding as fm
from paper_2606_11867_b200 import synth
from tests import gpu_common as G

pytestmark = pytest.mark.gpu


def _full_check(cfg, layers=None, mbs=None, what=""):
    ids, w, mb_off, se = G.make_case(cfg)
    ref = G.oracle_plan(ids, mb_off, se, cfg.E, cfg.P, cfg.Ns)
    assert ref["fault"] == 0
    sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se)
    assert sp.faults() == 0
    G.assert_plan_equal(sp, ref, what)
    layers = range(cfg.L) if layers is None else layers
    mbs = range(cfg.n_mb) if mbs is None else mbs
    x = G.activations(cfg, mb_off, mbs)
    G.check_data_path(sp, ref, x, layers, mbs, what)
    return sp, ref


def test_tiny_config1_everything(cuda_device):
    """BASELINE.json config 1 in full: E=8, top-2, 8 x 512 tokens, 4 ranks x (2+1), H=256 fp32."""
    _full_check(synth.config(1), what="cfg1")


@pytest.mark.parametrize("cfg_id,kw", [
    (2, dict(L=3, n_samples=12, sample_len=700, H=2048, mb_samples=4)),   # 2800 tok: ragged chunks
    (3, dict(L=2, n_samples=6, sample_len=1100, H=7168, mb_samples=2)),
    (5, dict(L=2, n_samples=3, sample_len=3000, H=4096, mb_samples=1)),   # K=10: 8-byte id rows
    (4, dict(L=2, n_samples=24, H=2048, mb_samples=5)),                   # lognormal lengths
    (4, dict(L=1, n_samples=9, H=512, mb_samples=1)),
])
def test_scaled_configs(cuda_device, cfg_id, kw):
    """Reduced copies of configs 2-5: several ranking chunks, ragged tails, every instance."""
    _full_check(synth.config(cfg_id).scaled(**kw), what=f"cfg{cfg_id}-scaled")


def test_ranged_calls_equal_per_instance(cuda_device):
    cfg = synth.config(2).scaled(L=2, n_samples=10, sample_len=333, H=256, mb_samples=3)
    ids, w, mb_off, se = G.make_case(cfg)
    ref = G.oracle_plan(ids, mb_off, se, cfg.E, cfg.P, cfg.Ns)
    sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se)
    s = sp.shape
    for (b, e) in [(0, cfg.n_mb), (1, 3), (2, 2)]:
        a_tok, b_tok = int(mb_off[b]), int(mb_off[e])
        n = b_tok - a_tok
        x = synth.gen_activations(cfg, max(n, 1), 99, G.DEV)
        perm = torch.full((max(n * s.K, 1),), -5, dtype=torch.int32, device=G.DEV)
        buf = torch.zeros((max(n * s.K, 1), s.H), dtype=s.act_torch_dtype, device=G.DEV)
        y = torch.zeros((max(n, 1), s.H), dtype=torch.float32, device=G.DEV)
        for l in range(cfg.L):
            sp.dispatch(l, b, e, x, perm, buf)
            sp.combine(l, b, e, buf, y)
            torch.cuda.synchronize()
            if n == 0:
                assert (perm == -5).all()
                continue
            perm_ref = ref["perm"][l, a_tok * s.K:b_tok * s.K]
            assert (perm[:n * s.K].cpu().numpy() == perm_ref).all()
            buf_ref = orc.gather(perm_ref, G.to_bits(x), s.K, pair_base=a_tok * s.K)
            assert (G.to_bits(buf)[:n * s.K] == buf_ref).all()
            y_ref = orc.combine(ref["inv"][l, a_tok:b_tok], w[l, a_tok:b_tok], buf_ref, s.act_dtype,
                                row_base=a_tok * s.K)
            assert (y[:n].cpu().numpy().view(np.uint32) == y_ref.view(np.uint32)).all()


def test_combine_identity_pins_on_gpu(cuda_device):
    """combine(dispatch(x)) with unit weights is exactly K*x; with w = 1/K exactly x (K = 8)."""
    cfg = synth.config(2).scaled(L=1, n_samples=2, sample_len=600, H=1024, mb_samples=2)
    ids, w, mb_off, se = G.make_case(cfg)
    for wval, scale in ((1.0, float(cfg.K)), (1.0 / cfg.K, 1.0)):
        sp = G.gpu_plan(fm.shape_of(cfg), ids, np.full_like(w, wval), mb_off, se)
        n = cfg.T
        x = synth.gen_activations(cfg, n, 5, G.DEV)
        buf = torch.empty((n * cfg.K, cfg.H), dtype=torch.bfloat16, device=G.DEV)
        y = torch.empty((n, cfg.H), dtype=torch.float32, device=G.DEV)
        sp.dispatch(0, 0, 1, x, None, buf)
        sp.combine(0, 0, 1, buf, y)
        assert torch.equal(y, x.float() * scale)


# ------------------------------------------------------------------ edge cases
_random_case = G.random_case


@pytest.mark.parametrize("seed", range(8))
def test_random_small_plans(cuda_device, seed):
    """Random placements with empty slots, same-rank duplicates, empty micro-steps, duplicate ids
    inside a token, K in {1,2,3,8,10,32,4,6}: every integer output equals the oracle."""
    rng = np.random.default_rng(1000 + seed)
    K = [1, 2, 3, 8, 10, 32, 4, 6][seed]
    E, P, Nr = [8, 16, 12, 64, 40, 64, 32, 24][seed], [2, 4, 3, 8, 5, 4, 8, 6][seed], [1, 2, 3, 2, 4, 0, 1, 2][seed]
    mb_sizes = [int(v) for v in rng.integers(0, 900, size=7)]
    mb_sizes[2] = 0
    mb_sizes[5] = 1
    ids, w, mb_off, se, Nb, Ns = _random_case(rng, 5, E, K, P, Nr, mb_sizes,
                                              dup_tokens=(seed % 2 == 1), skew=1.0 + 0.3 * seed)
    ref = G.oracle_plan(ids, mb_off, se, E, P, Ns)
    assert ref["fault"] == 0
    shape = fm.Shape(L=5, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=int(mb_off[-1]), n_mb=7, H=64,
                     act_dtype=fm.ACT_FP32)
    sp = G.gpu_plan(shape, ids, w, mb_off, se)
    assert sp.faults() == 0
    G.assert_plan_equal(sp, ref, f"random{seed}")
    x = {i: torch.randn((max(mb_sizes[i], 1), 64), device=G.DEV) for i in range(7)}
    G.check_data_path(sp, ref, x, range(5), range(7), f"random{seed}")


def test_quota_kernel_many_instances(cuda_device):
    """The quota kernel against the oracle's unit-by-unit rule on 2 x 128 x 6 random instances
    with many replicas: Phase B needs several passes and Phase C augmentations occur."""
    for (E, P, Nr, K, skew) in [(16, 8, 2, 2, 0.5), (32, 8, 4, 3, 0.8)]:
        rng = np.random.default_rng(7)
        L, mb_sizes = 128, [1, 2, 3, 4, 6, 100]
        n_mb = len(mb_sizes)
        ids, w, mb_off, se, Nb, Ns = _random_case(rng, L, E, K, P, Nr, mb_sizes, skew=skew)
        ref = G.oracle_plan(ids, mb_off, se, E, P, Ns)
        assert ref["fault"] == 0
        moved = passes = 0
        for i in range(n_mb):
            for l in range(L):
                _, _, _, (np_, mv), _ = orc.quota(ref["hist"][i, l], se[l], P, Ns)
                passes = max(passes, np_)
                moved += mv
        assert passes >= 3 and moved >= 5      # the cases exercise Phase B iteration and Phase C
        shape = fm.Shape(L=L, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=int(mb_off[-1]), n_mb=n_mb, H=8,
                         act_dtype=fm.ACT_FP32)
        sp = G.gpu_plan(shape, ids, w, mb_off, se)
        assert sp.faults() == 0
        G.assert_plan_equal(sp, ref, "quota-many")


def test_max_skew_single_expert(cuda_device):
    """Degenerate: every pair selects one of two experts (K=2), one of them replicated 3 times."""
    E, P, Nb, Nr, K, T = 8, 4, 2, 1, 2, 5000
    ids = np.zeros((1, T, K), dtype=np.int32)
    ids[0, :, 1] = 5
    se = np.array([[0, 1, 5, 2, 3, 5, 4, 5, -1, 6, 7, 5]], dtype=np.int32)
    mb_off = np.array([0, 4097, 5000], dtype=np.int32)
    w = np.ones((1, T, K), dtype=np.float32)
    ref = G.oracle_plan(ids, mb_off, se, E, P, Nb + Nr)
    sp = G.gpu_plan(fm.Shape(L=1, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=T, n_mb=2, H=8,
                             act_dtype=fm.ACT_FP32), ids, w, mb_off, se)
    assert sp.faults() == 0 and ref["fault"] == 0
    G.assert_plan_equal(sp, ref, "max-skew")
    x = {i: torch.randn((int(mb_off[i + 1] - mb_off[i]), 8), device=G.DEV) for i in range(2)}
    G.check_data_path(sp, ref, x, [0], [0, 1], "max-skew")


def test_expert_with_more_than_32_hosts(cuda_device):
    """One expert replicated on all 40 ranks (serial water-fill path), a second one on 20 ranks
    (warp path), the rest singly hosted."""
    rng = np.random.default_rng(11)
    E = P = 40
    Nb, Nr, K, L = 1, 2, 4, 3
    Ns = Nb + Nr
    mb_sizes = [700, 64, 3000]
    T = sum(mb_sizes)
    mb_off = np.concatenate([[0], np.cumsum(mb_sizes)]).astype(np.int32)
    p = np.full(E, 0.4 / (E - 2)); p[0] = 0.4; p[1] = 0.2
    g = rng.gumbel(size=(L, T, E)) + np.log(p)[None, None, :]
    ids = np.argsort(-g, axis=2)[:, :, :K].astype(np.int32)
    w = rng.random((L, T, K), dtype=np.float32)
    se = np.full((L, P * Ns), -1, dtype=np.int32)
    for l in range(L):
        for r in range(P):
            se[l, r * Ns] = r
            se[l, r * Ns + 1] = 0                      # expert 0 everywhere (rank 0: inactive duplicate)
            if r % 2 == 0:
                se[l, r * Ns + 2] = 1
    ref = G.oracle_plan(ids, mb_off, se, E, P, Ns)
    assert ref["fault"] == 0
    sp = G.gpu_plan(fm.Shape(L=L, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=T, n_mb=3, H=8,
                             act_dtype=fm.ACT_FP32), ids, w, mb_off, se)
    assert sp.faults() == 0
    G.assert_plan_equal(sp, ref, "40-hosts")


def test_per_microstep_placement(cuda_device):
    """placement_mb_stride = L*S: one placement per (micro-step, layer) (A^{(i)})."""
    rng = np.random.default_rng(3)
    L, n_mb, E, P, Nr, K = 2, 3, 16, 4, 2, 4
    mb_sizes = [300, 0, 1200]
    cases = [_random_case(rng, L, E, K, P, Nr, mb_sizes) for _ in range(n_mb)]
    ids, w, mb_off, _, Nb, Ns = cases[0]
    se = np.stack([c[3] for c in cases])                    # [n_mb, L, S]
    S = P * Ns
    shape = fm.Shape(L=L, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=int(mb_off[-1]), n_mb=n_mb, H=8,
                     act_dtype=fm.ACT_FP32, placement_mb_stride=L * S)
    sp = G.gpu_plan(shape, ids, w, mb_off, se)
    assert sp.faults() == 0
    hist, _, _ = orc.load_hist(ids, mb_off, E)
    for i in range(n_mb):
        a, b = int(mb_off[i]), int(mb_off[i + 1])
        for l in range(L):
            q, rl, so, _, f = orc.quota(hist[i, l], se[i, l], P, Ns)
            assert f == 0
            ps, inv, perm, f = orc.assign_instance(ids[l, a:b], se[i, l], q, so, E, base=a * K)
            assert f == 0
            assert (sp.quota[i, l].cpu().numpy() == q).all()
            assert (sp.rank_load[i, l].cpu().numpy() == rl).all()
            assert (sp.slot_off[i, l].cpu().numpy() == so).all()
            assert (sp.pair_slot[l, a:b].cpu().numpy().ravel() == ps).all()
            assert (sp.inv[l, a:b].cpu().numpy().ravel() == inv).all()


def test_caller_supplied_quota(cuda_device):
    """quota_in: a valid caller quota (here: everything on the LAST host of each expert) is
    honoured and validated by Eq.(8)/(9); an invalid one raises FAULT_QUOTA_IN."""
    cfg = synth.config(2).scaled(L=2, n_samples=4, sample_len=500, H=128, mb_samples=2)
    ids, w, mb_off, se = G.make_case(cfg)
    hist, _, _ = orc.load_hist(ids, mb_off, cfg.E)
    qin = np.zeros((cfg.n_mb, cfg.L, cfg.S), dtype=np.int32)
    for l in range(cfg.L):
        last = {int(e): j for j, e in enumerate(se[l]) if e >= 0}
        for e, j in last.items():
            qin[:, l, j] = hist[:, l, e]
    ref = G.oracle_plan(ids, mb_off, se, cfg.E, cfg.P, cfg.Ns, quota_in=qin)
    assert ref["fault"] == 0
    sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se, quota_in=qin)
    assert sp.faults() == 0
    G.assert_plan_equal(sp, ref, "quota_in")
    bad = qin.copy()
    j0 = int(np.argmax(bad[0, 0]))
    bad[0, 0, j0] -= 1
    sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se, quota_in=bad)
    assert sp.faults() & fm.FAULT_QUOTA_IN
    assert G.oracle_plan(ids, mb_off, se, cfg.E, cfg.P, cfg.Ns, quota_in=bad)["fault"] & orc.FAULT_QUOTA_IN


def test_device_faults(cuda_device):
    cfg = synth.config(1)
    ids, w, mb_off, se = G.make_case(cfg)
    shape = fm.shape_of(cfg)
    # id out of range: not counted, pair gets -1, other pairs still match the oracle
    bad_ids = ids.copy()
    bad_ids[0, 100, 1] = cfg.E + 3
    bad_ids[0, 700, 0] = -1
    ref = G.oracle_plan(bad_ids, mb_off, se, cfg.E, cfg.P, cfg.Ns)
    sp = G.gpu_plan(shape, bad_ids, w, mb_off, se)
    assert sp.faults() == fm.FAULT_ID_RANGE and ref["fault"] == orc.FAULT_ID_RANGE
    G.assert_plan_equal(sp, ref, "bad-id")
    # expert with tokens but no slot
    se2 = se.copy()
    victim = int(ids[0, 0, 0])
    se2[se2 == victim] = -1
    sp = G.gpu_plan(shape, ids, w, mb_off, se2)
    assert sp.faults() & fm.FAULT_NO_HOST
    assert (sp.inv.cpu().numpy() == -1).all() and (sp.quota.cpu().numpy() == 0).all()
    # slot_expert out of range
    se3 = se.copy()
    se3[0, 1] = cfg.E
    sp = G.gpu_plan(shape, ids, w, mb_off, se3)
    assert sp.faults() & fm.FAULT_SLOT_EXPERT
    # broken boundaries: histogram is all zero (as the oracle's), fault raised
    mb_bad = mb_off.copy()
    mb_bad[3] = mb_bad[2] - 1
    sp = G.gpu_plan(shape, ids, w, mb_bad, se)
    assert sp.faults() & fm.FAULT_MB_OFF
    assert (sp.hist.cpu().numpy() == 0).all()
    mb_bad = mb_off.copy()
    mb_bad[-1] -= 1
    sp = G.gpu_plan(shape, ids, w, mb_bad, se)
    assert sp.faults() & fm.FAULT_MB_OFF


def test_host_errors(cuda_device):
    cfg = synth.config(1)
    ids, w, mb_off, se = G.make_case(cfg)
    sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se)
    s = sp.shape
    import dataclasses
    with pytest.raises(fm.ForeMoEError) as ei:
        fm.workspace_bytes(dataclasses.replace(s, K=s.E + 1))
    assert ei.value.code == fm.ERR_INVALID_ARG
    with pytest.raises(fm.ForeMoEError) as ei:
        fm.workspace_bytes(dataclasses.replace(s, Nb=s.Nb + 1))
    assert ei.value.code == fm.ERR_INVALID_ARG
    with pytest.raises(fm.ForeMoEError) as ei:
        fm.workspace_bytes(dataclasses.replace(s, H=3))          # row bytes not a multiple of 16
    assert ei.value.code == fm.ERR_INVALID_ARG
    small = torch.empty(64, dtype=torch.uint8, device=G.DEV)
    with pytest.raises(fm.ForeMoEError) as ei:
        fm.assign(s, sp.ids, sp.mb_off, sp.hist, sp.slot_expert, None, sp.quota, sp.rank_load,
                  sp.slot_off, sp.pair_slot, sp.inv, small, sp.status)
    assert ei.value.code == fm.ERR_WORKSPACE
    x = torch.zeros((512, s.H), device=G.DEV)
    buf = torch.zeros((1024, s.H), device=G.DEV)
    with pytest.raises(fm.ForeMoEError) as ei:
        sp.dispatch(0, 3, 2, x, None, buf)
    assert ei.value.code == fm.ERR_INVALID_ARG
    with pytest.raises(fm.ForeMoEError) as ei:
        sp.dispatch(1, 0, 1, x, None, buf)                      # layer out of range
    assert ei.value.code == fm.ERR_INVALID_ARG
    with pytest.raises(fm.ForeMoEError) as ei:
        fm.dispatch(s, 0, 0, 1, sp.mb_off, sp.inv, x.view(-1)[1:].view(-1)[:511 * s.H].view(511, s.H),
                    None, buf)                                    # misaligned x
    assert ei.value.code == fm.ERR_INVALID_ARG


def test_step_host_matches_device_path(cuda_device):
    """foremoe_step_host (host buffers in, plan + last layer's y out) equals the device calls."""
    cfg = synth.config(2).scaled(L=3, n_samples=6, sample_len=400, H=256, mb_samples=2)
    ids, w, mb_off, se = G.make_case(cfg)
    s = fm.shape_of(cfg)
    ref = G.oracle_plan(ids, mb_off, se, cfg.E, cfg.P, cfg.Ns)
    pin = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).pin_memory()
    ids_h, w_h, mb_h, se_h = pin(ids, torch.int32), pin(w, torch.float32), pin(mb_off, torch.int32), pin(se, torch.int32)
    x_h = synth.gen_activations(cfg, cfg.T, 1, "cpu").pin_memory()
    q_h = torch.empty((s.n_mb, s.L, s.S), dtype=torch.int32).pin_memory()
    rl_h = torch.empty((s.n_mb, s.L, s.P), dtype=torch.int32).pin_memory()
    so_h = torch.empty((s.n_mb, s.L, s.S + 1), dtype=torch.int32).pin_memory()
    y_h = torch.empty((s.T, s.H), dtype=torch.float32).pin_memory()
    st_h = torch.full((1,), -1, dtype=torch.int32).pin_memory()
    arena = torch.empty(fm.step_host_arena_bytes(s, mb_h) + 256, dtype=torch.uint8, device=G.DEV)
    off = (-arena.data_ptr()) % 256
    fm.step_host(s, ids_h, w_h, mb_h, se_h, x_h, q_h, rl_h, so_h, y_h, arena[off:], st_h)
    assert int(st_h[0]) == 0
    assert (q_h.numpy() == ref["quota"]).all() and (rl_h.numpy() == ref["rank_load"]).all()
    assert (so_h.numpy() == ref["slot_off"]).all()
    l = s.L - 1
    xb = G.to_bits(x_h)
    for i in range(s.n_mb):
        a, b = int(mb_off[i]), int(mb_off[i + 1])
        buf_ref = orc.gather(ref["perm"][l, a * s.K:b * s.K], xb[a:b], s.K, pair_base=a * s.K)
        y_ref = orc.combine(ref["inv"][l, a:b], w[l, a:b], buf_ref, s.act_dtype, row_base=a * s.K)
        assert (y_h[a:b].numpy().view(np.uint32) == y_ref.view(np.uint32)).all()


def test_two_streams_reentrant(cuda_device):
    """The library is re-entrant per stream: independent instances issued on two non-default streams
    (each with its own buffers) give the results of the sequential default-stream calls, bit for bit."""
    cfg = synth.config(2).scaled(L=2, n_samples=12, sample_len=500, H=512, mb_samples=3)
    ids, w, mb_off, se = G.make_case(cfg)
    sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se)
    s = sp.shape
    x = G.activations(cfg, mb_off, range(cfg.n_mb))
    inst = [(l, i) for l in range(cfg.L) for i in range(cfg.n_mb)]
    n_max = max(int(mb_off[i + 1] - mb_off[i]) for i in range(cfg.n_mb))

    def bufs():
        return (torch.zeros((n_max * s.K,), dtype=torch.int32, device=G.DEV),
                torch.zeros((n_max * s.K, s.H), dtype=s.act_torch_dtype, device=G.DEV),
                torch.zeros((n_max, s.H), dtype=torch.float32, device=G.DEV))

    ref_out = {}
    perm, buf, y = bufs()
    for (l, i) in inst:
        sp.dispatch(l, i, i + 1, x[i], perm, buf)
        sp.combine(l, i, i + 1, buf, y)
        torch.cuda.synchronize()
        ref_out[(l, i)] = (perm.clone(), buf.clone(), y.clone())
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    got = {}
    torch.cuda.synchronize()
    for j, st in enumerate(streams):
        with torch.cuda.stream(st):
            for (l, i) in inst[j::2]:
                p_, b_, y_ = bufs()
                sp.dispatch(l, i, i + 1, x[i], p_, b_)
                sp.combine(l, i, i + 1, b_, y_)
                got[(l, i)] = (p_, b_, y_)
    torch.cuda.synchronize()
    for key in inst:
        n = int(mb_off[key[1] + 1] - mb_off[key[1]])
        for a, b in zip(ref_out[key], got[key]):
            rows = n * s.K if a.shape[0] == n_max * s.K else n
            assert torch.equal(a[:rows].view(torch.uint8), b[:rows].view(torch.uint8)), key


def test_two_host_threads_two_streams(cuda_device):
    """Two HOST threads, each driving its own stream with its own shape (so each needs different
    kernel variants and launch facts), started together on variants no earlier call has prepared:
    results equal the sequential ones bit for bit (the launch-fact memo is lock-free and per device)."""
    import threading
    cases = []
    for (H, K, E, P, Nr, seed) in [(1544, 8, 64, 8, 2, 1), (776, 6, 24, 6, 2, 2)]:
        rng = np.random.default_rng(900 + seed)
        mb_sizes = [400, 33, 800]
        ids, w, mb_off, se, Nb, Ns = G.random_case(rng, 2, E, K, P, Nr, mb_sizes)
        shape = fm.Shape(L=2, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=int(mb_off[-1]), n_mb=3, H=H,
                         act_dtype=fm.ACT_BF16)
        sp = G.gpu_plan(shape, ids, w, mb_off, se)
        x = {i: torch.randn((mb_sizes[i], H), device=G.DEV).bfloat16() for i in range(3)}
        cases.append((sp, mb_sizes, x))

    def run_all(sp, mb_sizes, x, out):
        s = sp.shape
        for rep in range(4):
            for l in range(2):
                for i in range(3):
                    n = mb_sizes[i]
                    perm = torch.empty((n * s.K,), dtype=torch.int32, device=G.DEV)
                    buf = torch.empty((n * s.K, s.H), dtype=torch.bfloat16, device=G.DEV)
                    y = torch.empty((n, s.H), dtype=torch.float32, device=G.DEV)
                    dx = torch.empty((n, s.H), dtype=torch.float32, device=G.DEV)
                    sp.dispatch(l, i, i + 1, x[i], perm, buf)
                    sp.combine(l, i, i + 1, buf, y)
                    sp.dispatch_bwd(l, i, i + 1, buf, dx)
                    out[(rep, l, i)] = (perm, buf, y, dx)

    errors = []

    def worker(case, out):
        try:
            torch.cuda.set_device(0)
            with torch.cuda.stream(torch.cuda.Stream()):
                run_all(*case, out)
                torch.cuda.current_stream().synchronize()
        except Exception as e:      # surfaced below
            errors.append(e)

    outs = [dict(), dict()]
    threads = [threading.Thread(target=worker, args=(c, o)) for c, o in zip(cases, outs)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    torch.cuda.synchronize()
    for case, got in zip(cases, outs):
        ref = {}
        run_all(*case, ref)
        torch.cuda.synchronize()
        for key in ref:
            for a, b in zip(ref[key], got[key]):
                assert torch.equal(a.view(torch.uint8), b.view(torch.uint8)), key
        assert case[0].faults() == 0


_CAPTURE_FIRST_CALL = r"""
import sys, numpy as np, torch
sys.path.insert(0, sys.argv[1])
from paper_2606_11867_b200 import binding as fm, synth
from tests import gpu_common as G
cfg = synth.config(2).scaled(L=1, n_samples=6, sample_len=400, H=512, mb_samples=3)
ids, w, mb_off, se = G.make_case(cfg)
sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se)      # plan kernels only
s = sp.shape
n = int(mb_off[1] - mb_off[0])
x = synth.gen_activations(cfg, n, 0, G.DEV)
dy = torch.randn((n, s.H), device=G.DEV)
mk = lambda: (torch.zeros((n * s.K,), dtype=torch.int32, device=G.DEV),
              torch.zeros((n * s.K, s.H), dtype=s.act_torch_dtype, device=G.DEV),
              torch.zeros((n, s.H), dtype=torch.float32, device=G.DEV),
              torch.zeros((n * s.K, s.H), dtype=s.act_torch_dtype, device=G.DEV),
              torch.zeros((n, s.H), dtype=torch.float32, device=G.DEV),
              torch.zeros((s.L, s.T, s.K), dtype=torch.float32, device=G.DEV),
              torch.zeros((n * s.K, s.H), dtype=s.act_torch_dtype, device=G.DEV))
def run(b):
    perm, buf, y, d_buf, dx, dw, d_buf2 = b
    sp.dispatch(0, 0, 1, x, perm, buf)
    sp.combine(0, 0, 1, buf, y)
    sp.combine_bwd(0, 0, 1, dy, buf, d_buf, dw)
    sp.combine_bwd(0, 0, 1, dy, None, d_buf2, None)
    sp.dispatch_bwd(0, 0, 1, d_buf, dx)
fm.warmup(s)                        # no data-path call has run in this process
graphed = mk()
torch.cuda.synchronize()
g = torch.cuda.CUDAGraph()
with torch.cuda.graph(g):
    run(graphed)                    # the FIRST data-path calls of the process, under capture
g.replay()
torch.cuda.synchronize()
eager = mk()
run(eager)
torch.cuda.synchronize()
for a, b in zip(eager, graphed):
    assert torch.equal(a.view(torch.uint8), b.view(torch.uint8))
assert sp.faults() == 0
print("capture-first-call ok")
"""


def test_graph_capture_of_first_call_after_warmup(cuda_device):
    """foremoe_warmup makes the data-path calls capturable from the very first call: a fresh process
    warms up, captures dispatch + combine + both backward calls without ever running them eagerly,
    replays, and the results equal the eager calls made afterwards."""
    import os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", _CAPTURE_FIRST_CALL, root], capture_output=True, text=True,
                       cwd=root, timeout=600)
    assert r.returncode == 0 and "capture-first-call ok" in r.stdout, (r.stdout[-2000:], r.stderr[-4000:])


_CAPTURE_TWO_SHAPES = r"""
import dataclasses, sys, numpy as np, torch
sys.path.insert(0, sys.argv[1])
from paper_2606_11867_b200 import binding as fm, synth
from tests import gpu_common as G
base = synth.config(2).scaled(L=1, n_samples=4, sample_len=300, H=1024, mb_samples=2)
plans = []
for K in (3, 5, 7):          # no kernel is specialised for these K: the three shapes share the generic
    cfg = dataclasses.replace(base, K=K)          # instantiations and differ only in shared-memory size
    ids, w, mb_off, se = G.make_case(cfg)
    sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se)
    n = int(mb_off[1] - mb_off[0])
    plans.append((sp, n, synth.gen_activations(cfg, n, 0, G.DEV), torch.randn((n, cfg.H), device=G.DEV)))
def mk(sp, n):
    s = sp.shape
    return (torch.zeros((n * s.K,), dtype=torch.int32, device=G.DEV),
            torch.zeros((n * s.K, s.H), dtype=s.act_torch_dtype, device=G.DEV),
            torch.zeros((n, s.H), dtype=torch.float32, device=G.DEV),
            torch.zeros((n * s.K, s.H), dtype=s.act_torch_dtype, device=G.DEV),
            torch.zeros((n, s.H), dtype=torch.float32, device=G.DEV),
            torch.zeros((s.L, s.T, s.K), dtype=torch.float32, device=G.DEV))
def run(sp, x, dy, b):
    perm, buf, y, d_buf, dx, dw = b
    sp.dispatch(0, 0, 1, x, perm, buf)
    sp.combine(0, 0, 1, buf, y)
    sp.combine_bwd(0, 0, 1, dy, buf, d_buf, dw)
    sp.dispatch_bwd(0, 0, 1, d_buf, dx)
for sp, n, x, dy in plans:
    fm.warmup(sp.shape)          # all three warmed BEFORE anything is captured
graphed = [mk(sp, n) for sp, n, x, dy in plans]
torch.cuda.synchronize()
g = torch.cuda.CUDAGraph()
with torch.cuda.graph(g):
    for (sp, n, x, dy), b in zip(plans, graphed):
        run(sp, x, dy, b)        # first data-path calls of the process, first shape first
g.replay()
torch.cuda.synchronize()
for (sp, n, x, dy), b in zip(plans, graphed):
    e = mk(sp, n)
    run(sp, x, dy, e)
    torch.cuda.synchronize()
    for u, v in zip(e, b):
        assert torch.equal(u.view(torch.uint8), v.view(torch.uint8))
    assert sp.faults() == 0
print("capture-two-shapes ok")
"""


def test_graph_capture_after_warming_several_shapes(cuda_device):
    """Warming a second and third shape that select the same kernel instantiations must not push the
    first shape's launch facts out of the per-device memo: all three are then captured from their very
    first call (a miss would query occupancy / set the shared-memory attribute during capture).  The memo
    itself is checked on the host by tests/test_abi.py (memo_check.cu); this is the end-to-end use."""
    import os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", _CAPTURE_TWO_SHAPES, root], capture_output=True, text=True,
                       cwd=root, timeout=600)
    assert r.returncode == 0 and "capture-two-shapes ok" in r.stdout, (r.stdout[-2000:], r.stderr[-4000:])


def test_cuda_graph_replay(cuda_device):
    """The data-path calls are capturable into a CUDA graph once each kernel variant has run eagerly
    (the first launch of a variant queries occupancy / opts into large shared memory); the replay
    reproduces the eager results bit for bit, forward and backward."""
    cfg = synth.config(2).scaled(L=1, n_samples=6, sample_len=400, H=512, mb_samples=3)
    ids, w, mb_off, se = G.make_case(cfg)
    sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se)
    s = sp.shape
    n = int(mb_off[1] - mb_off[0])
    x = synth.gen_activations(cfg, n, 0, G.DEV)
    dy = torch.randn((n, s.H), device=G.DEV)
    mk = lambda: (torch.zeros((n * s.K,), dtype=torch.int32, device=G.DEV),
                  torch.zeros((n * s.K, s.H), dtype=s.act_torch_dtype, device=G.DEV),
                  torch.zeros((n, s.H), dtype=torch.float32, device=G.DEV),
                  torch.zeros((n * s.K, s.H), dtype=s.act_torch_dtype, device=G.DEV),
                  torch.zeros((n, s.H), dtype=torch.float32, device=G.DEV),
                  torch.zeros((s.L, s.T, s.K), dtype=torch.float32, device=G.DEV))

    def run(b):
        perm, buf, y, d_buf, dx, dw = b
        sp.dispatch(0, 0, 1, x, perm, buf)
        sp.combine(0, 0, 1, buf, y)
        sp.combine_bwd(0, 0, 1, dy, buf, d_buf, dw)
        sp.dispatch_bwd(0, 0, 1, d_buf, dx)

    eager = mk()
    run(eager)                                   # also the warm-up of every kernel variant
    torch.cuda.synchronize()
    graphed = mk()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        run(graphed)
    for t in graphed:
        t.zero_()
    g.replay()
    g.replay()
    torch.cuda.synchronize()
    for a, b in zip(eager, graphed):
        assert torch.equal(a.view(torch.uint8), b.view(torch.uint8))


def test_empty_step(cuda_device):
    """T = 0 (a step without tokens): foremoe_plan and load_hist + assign give the all-zero plan of the
    oracle, and the data-path calls on the empty range are no-ops."""
    rng = np.random.default_rng(5)
    L, E, K, P, Nr = 2, 16, 2, 4, 1
    ids, w, mb_off, se, Nb, Ns = G.random_case(rng, L, E, K, P, Nr, [0, 0, 0])
    shape = fm.Shape(L=L, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=0, n_mb=3, H=64, act_dtype=fm.ACT_FP32)
    ref = G.oracle_plan(ids, mb_off, se, E, P, Ns)
    sp = G.gpu_plan(shape, ids, w, mb_off, se)
    assert sp.faults() == 0 and ref["fault"] == 0
    for name in ("hist", "step_hist", "quota", "rank_load", "slot_off"):
        got = getattr(sp, name).cpu().numpy()
        assert (got == ref[name]).all() and (got == 0).all(), name
    x = torch.zeros((1, shape.H), device=G.DEV)
    buf = torch.full((1, shape.H), 7.0, device=G.DEV)
    y = torch.full((1, shape.H), 7.0, device=G.DEV)
    sp.dispatch(0, 0, 3, x, None, buf)
    sp.combine(1, 1, 2, buf, y)
    torch.cuda.synchronize()
    assert (buf == 7.0).all() and (y == 7.0).all()


@pytest.mark.parametrize("E,P,Nr", [(64, 8, 2), (512, 32, 4), (1024, 32, 8)])
def test_quota_kernel_index_width(cuda_device, E, P, Nr):
    """k_quota holds its index tables as int32 for small shapes and as int16 once shared memory would cap
    the resident CTAs (E = 512 and up here): the same random plans, heavy replication, both against O2."""
    rng = np.random.default_rng(E)
    L, K = 2, 4
    ids, w, mb_off, se, Nb, Ns = G.random_case(rng, L, E, K, P, Nr, [300, 0, 777, 64], skew=1.3,
                                               empty_slots=False, same_rank_dup=False)
    # replicate the hottest experts many times so that Phase B iterates
    step = orc.load_hist(ids, mb_off, E)[1]
    for l in range(L):
        hot = np.argsort(-step[l])[:max(2, P // 4)]
        for r in range(P):
            for a in range(Nr):
                se[l, r * Ns + Nb + a] = hot[(r + a) % len(hot)]
    shape = fm.Shape(L=L, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=int(mb_off[-1]), n_mb=4, H=64, act_dtype=fm.ACT_FP32)
    ref = G.oracle_plan(ids, mb_off, se, E, P, Ns)
    assert ref["fault"] == 0
    sp = G.gpu_plan(shape, ids, w, mb_off, se)
    assert sp.faults() == 0
    G.assert_plan_equal(sp, ref, f"index-width E={E}")


@pytest.mark.parametrize("seed", [1, 2])
def test_fuzz_shapes(cuda_device, seed):
    """400 random shapes per seed (P from 1 to 64, Nb from 1 to 16 incl. non powers of two, K from 1 to 32, Nr
    from 0 to 5, empty micro-steps, duplicate ids in a token, one expert replicated on every rank): the plan
    by foremoe_plan and by load_hist + assign against the oracle, every output."""
    rng = np.random.default_rng(seed)
    for _ in range(400):
        P = int(rng.choice([1, 2, 3, 4, 8, 16, 32, 64]))
        Nb = int(rng.choice([1, 2, 3, 4, 7, 16]))
        E = P * Nb
        K = int(rng.integers(1, min(E, 32) + 1))
        Nr = int(rng.choice([0, 1, 2, 5]))
        L = int(rng.integers(1, 4))
        n_mb = int(rng.integers(1, 6))
        sizes = [int(rng.choice([0, 1, 7, 100, 513, 3000])) for _ in range(n_mb)]
        if sum(sizes) * K > 60000:
            sizes = [min(s, 400) for s in sizes]
        ids, w, mb_off, se, _, Ns = G.random_case(rng, L, E, K, P, Nr, sizes, dup_tokens=bool(rng.integers(2)),
                                                  skew=float(rng.choice([0.0, 1.0, 2.5])))
        if rng.random() < 0.3 and Nr:
            for l in range(L):
                for r in range(P):
                    se[l, r * Ns + Nb] = se[l, 0]
        shape = fm.Shape(L=L, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=int(mb_off[-1]), n_mb=n_mb, H=8, act_dtype=fm.ACT_FP32)
        ref = G.oracle_plan(ids, mb_off, se, E, P, Ns)
        sp = G.gpu_plan(shape, ids, w, mb_off, se)
        assert sp.faults() == ref["fault"], (shape, sp.faults(), ref["fault"])
        if ref["fault"] == 0:
            G.assert_plan_equal(sp, ref, str(shape))


def test_fuzz_data_path_shapes(cuda_device):
    """250 random data-path shapes (K from 1 to 32, rows from 16 bytes to 7 KB incl. sizes that are no
    multiple of the kernels' slices, bf16 and fp32, empty and tiny micro-steps, both stream-order modes):
    perm / buf bit-exact and y bit-identical against O5 / O6, also on expert outputs that differ per k."""
    rng = np.random.default_rng(77)
    done = 0
    while done < 250:
        P = int(rng.choice([1, 2, 4, 8]))
        Nb = int(rng.choice([1, 2, 4, 16]))
        E = P * Nb
        K = int(rng.choice([k for k in (1, 2, 3, 4, 5, 6, 8, 10, 16, 32) if k <= E]))
        Nr, L, n_mb = int(rng.choice([0, 1, 2])), int(rng.integers(1, 3)), int(rng.integers(1, 4))
        bf16 = bool(rng.integers(2))
        H = (8 if bf16 else 4) * int(rng.choice([1, 2, 3, 8, 31, 64, 65, 128, 256, 257, 896, 1024, 1792]))
        sizes = [int(rng.choice([0, 1, 5, 33, 200, 700])) for _ in range(n_mb)]
        while sum(sizes) * K * H > 6_000_000:
            sizes = [s // 2 for s in sizes]
        ids, w, mb_off, se, _, Ns = G.random_case(rng, L, E, K, P, Nr, sizes, skew=float(rng.choice([0.0, 1.5])))
        shape = fm.Shape(L=L, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=int(mb_off[-1]), n_mb=n_mb, H=H,
                         act_dtype=fm.ACT_BF16 if bf16 else fm.ACT_FP32, flags=int(rng.integers(2)))
        if shape.T == 0:
            continue
        ref = G.oracle_plan(ids, mb_off, se, E, P, Ns)
        if ref["fault"]:
            continue
        sp = G.gpu_plan(shape, ids, w, mb_off, se)
        G.assert_plan_equal(sp, ref, str(shape))
        x = {i: torch.randn(max(int(mb_off[i + 1] - mb_off[i]), 1), H, device=G.DEV).to(shape.act_torch_dtype)
             for i in range(n_mb)}
        G.check_data_path(sp, ref, x, range(L), range(n_mb), str(shape))
        done += 1


def test_quota_only_assign_takes_no_ids(cuda_device):
    """foremoe_assign with pair_slot = inv = NULL computes the quotas only and does not read the ids
    (include/foremoe.h): ids = NULL is accepted and gives the quotas of the full call."""
    cfg = synth.config(2).scaled(L=2, n_samples=6, sample_len=500, H=256, mb_samples=2)
    ids, w, mb_off, se = G.make_case(cfg)
    sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se)
    q, rl, so = (torch.full_like(t, -9) for t in (sp.quota, sp.rank_load, sp.slot_off))
    fm.assign(sp.shape, None, sp.mb_off, sp.hist, sp.slot_expert, None, q, rl, so, None, None, sp.workspace, sp.status)
    torch.cuda.synchronize()
    assert torch.equal(q, sp.quota) and torch.equal(rl, sp.rank_load) and torch.equal(so, sp.slot_off)
    assert sp.faults() == 0
    with pytest.raises(fm.ForeMoEError):           # assigning the pairs does need them
        fm.assign(sp.shape, None, sp.mb_off, sp.hist, sp.slot_expert, None, q, rl, so, sp.pair_slot, sp.inv,
                  sp.workspace, sp.status)


def test_data_path_without_torchs_raw_stream_getter(cuda_device, monkeypatch):
    """binding.DataPath on a torch build that lacks torch._C._cuda_getCurrentRawStream: the public
    current_stream() is used instead, on a side stream too, with the same results."""
    cfg = synth.config(2).scaled(L=1, n_samples=4, sample_len=300, H=512, mb_samples=2)
    ids, w, mb_off, se = G.make_case(cfg)
    sp = G.gpu_plan(fm.shape_of(cfg), ids, w, mb_off, se)
    s, n = sp.shape, int(mb_off[1] - mb_off[0])
    x = synth.gen_activations(cfg, n, 0, G.DEV)
    mk = lambda: (torch.zeros((n * s.K,), dtype=torch.int32, device=G.DEV),
                  torch.zeros((n * s.K, s.H), dtype=s.act_torch_dtype, device=G.DEV),
                  torch.zeros((n, s.H), dtype=torch.float32, device=G.DEV))
    ref = mk()
    sp.dispatch(0, 0, 1, x, ref[0], ref[1])
    sp.combine(0, 0, 1, ref[1], ref[2])
    torch.cuda.synchronize()
    monkeypatch.setattr(fm, "_raw_stream", None)
    got = mk()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        assert fm._stream_on(0) == side.cuda_stream == fm._stream()
        sp.dispatch(0, 0, 1, x, got[0], got[1])
        sp.combine(0, 0, 1, got[1], got[2])
    torch.cuda.synchronize()
    for a, b in zip(ref, got):
        assert torch.equal(a.view(torch.uint8), b.view(torch.uint8))
