"""GPU parity of foremoe_combine (a6) on expert outputs that DIFFER per k, and of the un-synchronised
assign -> dispatch -> combine pipeline.

PAPER.md:56 sec. 2.1 defines the combine on the selected experts' outputs ("the weighted sum of the
selected experts' outputs").  With the identity expert (expert_out = buf) the K rows a token reads
are bit-identical, so a kernel that pairs w[t][k] with the row of inv[t][k'] would still pass; the
cases here feed independent random rows in slot order and compare y with O6 bit for bit, for every
K specialisation of the ring kernel, the generic-K path, bf16 and fp32, ragged rows, faulted pairs
(inv < 0) and ranged calls.
"""
import numpy as np
import pytest
import torch

from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import binding as fm
from paper_2606_11867_b200 import runner, synth
from tests import gpu_common as G

pytestmark = pytest.mark.gpu

# (K, E, P, Nr): every K_T specialisation (2, 4, 6, 8, 10) and the generic path (1, 3, 5, 32)
K_CASES = [(1, 8, 2, 1), (2, 16, 4, 2), (3, 12, 3, 1), (4, 32, 8, 1), (5, 20, 4, 2), (6, 24, 6, 2),
           (8, 64, 8, 2), (10, 40, 5, 4), (32, 64, 4, 1)]


@pytest.mark.parametrize("K,E,P,Nr", K_CASES)
@pytest.mark.parametrize("act", [fm.ACT_BF16, fm.ACT_FP32])
def test_combine_random_rows(cuda_device, K, E, P, Nr, act):
    """Random expert outputs, non-uniform weights, H chosen so that rows are whole 512-byte slices
    (H = 1024 bf16 / 512 fp32), a ragged last slice, and a row shorter than one slice."""
    rng = np.random.default_rng(4000 + 37 * K + act)
    mb_sizes = [257, 0, 1, 1300, 64]
    L = 2
    ids, w, mb_off, se, Nb, Ns = G.random_case(rng, L, E, K, P, Nr, mb_sizes, skew=1.2,
                                               same_rank_dup=False, empty_slots=False)
    w = (w * 2.0 - 0.7).astype(np.float32)                 # both signs, not normalised
    ref = G.oracle_plan(ids, mb_off, se, E, P, Ns)
    assert ref["fault"] == 0
    es = 2 if act == fm.ACT_BF16 else 4
    for H in (2048 // es, 2064 // es * 1, 1360 // es, 400 // es):
        shape = fm.Shape(L=L, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=int(mb_off[-1]), n_mb=len(mb_sizes),
                         H=H, act_dtype=act)
        sp = G.gpu_plan(shape, ids, w, mb_off, se)
        assert sp.faults() == 0
        for l in range(L):
            for i in range(len(mb_sizes)):
                a, b = int(mb_off[i]), int(mb_off[i + 1])
                G.check_combine_random(sp, ref["inv"][l, a:b], w[l, a:b], l, i, a, b - a,
                                       seed=K * 100 + l * 10 + i, what=f"K={K} H={H} act={act}")


@pytest.mark.parametrize("act", [fm.ACT_BF16, fm.ACT_FP32])
def test_combine_random_rows_ranged_and_faulted(cuda_device, act):
    """A ranged call over several micro-steps (one empty) and pairs with inv < 0 (ids out of range):
    a faulted pair contributes nothing, even when the rows it would have read hold NaN / Inf."""
    rng = np.random.default_rng(77 + act)
    K, E, P, Nr, L = 8, 32, 4, 2, 2
    mb_sizes = [300, 0, 5, 700, 129, 1]
    ids, w, mb_off, se, Nb, Ns = G.random_case(rng, L, E, K, P, Nr, mb_sizes, skew=1.0)
    T = int(mb_off[-1])
    bad = rng.choice(T * K, size=40, replace=False)
    ids.reshape(L, -1)[0, bad] = E + 5
    ids.reshape(L, -1)[1, bad[:7]] = -3
    ids[0, 10, :] = -1                                       # a token with no valid pair at all: y = 0
    ref = G.oracle_plan(ids, mb_off, se, E, P, Ns)
    assert ref["fault"] == orc.FAULT_ID_RANGE
    H = 1096 if act == fm.ACT_BF16 else 548                  # ragged: 2192 bytes per row
    shape = fm.Shape(L=L, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=T, n_mb=len(mb_sizes), H=H, act_dtype=act)
    sp = G.gpu_plan(shape, ids, w, mb_off, se)
    assert sp.faults() == fm.FAULT_ID_RANGE
    G.assert_plan_equal(sp, ref, "faulted")
    for (b, e) in [(0, len(mb_sizes)), (2, 5), (3, 4), (1, 2)]:
        a_tok, b_tok = int(mb_off[b]), int(mb_off[e])
        n = b_tok - a_tok
        if n == 0:
            continue
        eo = G.random_expert_out(n * K, H, shape.act_torch_dtype, seed=b * 10 + e)
        # rows no valid pair maps to: poison (a skipped pair must not read them into the sum)
        used = np.zeros(n * K, dtype=bool)
        for l in range(L):
            iv = ref["inv"][l, a_tok:b_tok].ravel()
            used[iv[iv >= 0] - a_tok * K] = True
        eo[torch.from_numpy(~used).to(G.DEV)] = float("nan")
        eo[0, :] = eo[0, :]                                  # keep contiguous
        for l in range(L):
            G.check_combine_random(sp, ref["inv"][l, a_tok:b_tok], w[l, a_tok:b_tok], l, b, a_tok, n,
                                   seed=0, what=f"ranged[{b},{e})", mb_end=e, eo=eo)
    # the token without a valid pair sums nothing
    y = torch.full((mb_sizes[0], H), float("nan"), dtype=torch.float32, device=G.DEV)
    sp.combine(0, 0, 1, G.random_expert_out(mb_sizes[0] * K, H, shape.act_torch_dtype, 3), y)
    assert (y[10] == 0).all()


def test_dispatch_bwd_and_combine_share_pairing(cuda_device):
    """w == 1 for one k and 0 elsewhere selects exactly row inv[t][k]: y == float(expert_out[inv[t][k]])
    for every k in turn (the most direct statement of the w_k <-> row pairing)."""
    rng = np.random.default_rng(5)
    K, E, P, Nr = 8, 64, 8, 2
    ids, w, mb_off, se, Nb, Ns = G.random_case(rng, 1, E, K, P, Nr, [777], skew=1.1)
    ref = G.oracle_plan(ids, mb_off, se, E, P, Ns)
    shape = fm.Shape(L=1, E=E, K=K, P=P, Nb=Nb, Nr=Nr, T=777, n_mb=1, H=2048, act_dtype=fm.ACT_BF16)
    eo = G.random_expert_out(777 * K, 2048, torch.bfloat16, 9)
    inv = torch.from_numpy(ref["inv"][0].astype(np.int64)).to(G.DEV)
    for k in range(K):
        wk = np.zeros_like(w)
        wk[0, :, k] = 1.0
        sp = G.gpu_plan(shape, ids, wk, mb_off, se)
        y = torch.empty((777, 2048), dtype=torch.float32, device=G.DEV)
        sp.combine(0, 0, 1, eo, y)
        # 0 * v + ... : signed zeros aside, the selected row comes back exactly
        assert torch.equal(y, eo[inv[:, k]].float() + 0.0), k


@pytest.mark.parametrize("flags", [0, fm.FLAG_PLAN_STABLE])
def test_unsynchronised_pipeline_replan(cuda_device, flags):
    """load_hist -> assign -> dispatch -> combine enqueued on one stream with NO synchronise in
    between, after the same buffers held the plan of a DIFFERENT trace: the data-path kernels must
    see the new inv.  They are launched with programmatic stream serialisation; by default they read
    nothing before their grid-dependency wait, and with FOREMOE_FLAG_PLAN_STABLE they may read the
    plan arrays early -- which is still covered right after foremoe_assign, because it ends with a
    full serialisation point.  Compared with the oracle for the second trace, bit for bit."""
    cfg = synth.config(2).scaled(L=2, n_samples=8, sample_len=900, H=2048, mb_samples=4)
    ids_a, w_a, mb_off, se = G.make_case(cfg)
    cfg_b = synth.config(2).scaled(L=2, n_samples=8, sample_len=900, H=2048, mb_samples=4)
    cfg_b.seed = cfg.seed + 12345
    ids_b, w_b, mb_off_b, _ = G.make_case(cfg_b)
    assert (mb_off_b == mb_off).all() and (ids_a != ids_b).any()
    ref = G.oracle_plan(ids_b, mb_off, se, cfg.E, cfg.P, cfg.Ns)
    assert ref["fault"] == 0
    s = fm.shape_of(cfg, flags=flags)
    t = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).to(G.DEV)
    ids_d, w_d = t(ids_a, torch.int32), t(w_a, torch.float32)
    ids_bd, w_bd = t(ids_b, torch.int32), t(w_b, torch.float32)
    sp = runner.StepPlan(s, ids_d, w_d, t(mb_off, torch.int32), t(se, torch.int32))
    n = [int(mb_off[i + 1] - mb_off[i]) for i in range(cfg.n_mb)]
    x = G.activations(cfg, mb_off, range(cfg.n_mb))
    out = {(l, i): (torch.full((n[i] * s.K,), -5, dtype=torch.int32, device=G.DEV),
                    torch.zeros((n[i] * s.K, s.H), dtype=torch.bfloat16, device=G.DEV),
                    torch.full((n[i], s.H), float("nan"), dtype=torch.float32, device=G.DEV))
           for l in range(cfg.L) for i in range(cfg.n_mb)}
    for rep in range(3):
        sp.plan()                                   # plan of trace A lands in hist / quota / inv
        torch.cuda.synchronize()
        ids_d.copy_(ids_bd)                         # stream-ordered: same buffers, trace B
        w_d.copy_(w_bd)
        sp.plan()                                   # re-plan, then the data path, no sync anywhere
        for (l, i), (perm, buf, y) in out.items():
            sp.dispatch(l, i, i + 1, x[i], perm, buf)
            sp.combine(l, i, i + 1, buf, y)
        torch.cuda.synchronize()
        assert sp.faults() == 0
        G.assert_plan_equal(sp, ref, "replan")
        for (l, i), (perm, buf, y) in out.items():
            a, b = int(mb_off[i]), int(mb_off[i + 1])
            perm_ref = ref["perm"][l, a * s.K:b * s.K]
            assert (perm.cpu().numpy() == perm_ref).all(), ("perm", rep, l, i)
            buf_ref = orc.gather(perm_ref, G.to_bits(x[i]), s.K, pair_base=a * s.K)
            assert (G.to_bits(buf) == buf_ref).all(), ("buf", rep, l, i)
            y_ref = orc.combine(ref["inv"][l, a:b], w_b[l, a:b], buf_ref, s.act_dtype, row_base=a * s.K)
            assert (y.cpu().numpy().view(np.uint32) == y_ref.view(np.uint32)).all(), ("y", rep, l, i)
        ids_d.copy_(t(ids_a, torch.int32))
        w_d.copy_(t(w_a, torch.float32))
