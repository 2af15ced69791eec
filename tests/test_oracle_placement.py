"""Pins for the placement oracles O7 (Stage 1 rank-level LPT, Alg. 1) and O8
(Alg. 3 Stages 2-3): a hand-worked vector, closed forms, the greedy invariants
checked from the OUTPUT alone, Eq.(6)/(7) structure, and the effect on Stage 4's max rank load."""
import json
import os

import numpy as np
import pytest

from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import synth

HERE = os.path.dirname(os.path.abspath(__file__))


def _structure_ok(se, E, P, Nb, Nr, c=None, base_only=False):
    Ns = Nb + Nr
    se = se.reshape(P, Ns)
    base = se[:, :Nb]
    # Eq.(7) coverage + one base slot per expert; base slots filled front to back
    ids, cnt = np.unique(base[base >= 0], return_counts=True)
    assert (cnt == 1).all() and len(ids) == E
    for r in range(P):
        row = base[r]
        k = int((row >= 0).sum())
        assert (row[:k] >= 0).all() and (row[k:] == -1).all()
        red = se[r, Nb:]
        k = int((red >= 0).sum())
        assert (red[:k] >= 0).all() and (red[k:] == -1).all()
        live = se[r][se[r] >= 0]
        assert len(set(live.tolist())) == len(live)          # never twice on one rank
    if base_only:
        assert (se[:, Nb:] == -1).all()
    if c is not None:                                        # zero-load experts are never replicated
        for e in se[:, Nb:].ravel():
            assert e < 0 or c[e] > 0


def test_golden_vector():
    g = json.load(open(os.path.join(HERE, "golden", "placement_vectors.json")))
    c = np.array(g["c"])
    se, f = orc.base_placement(c, g["P"], g["Nb"], g["Nr"])
    assert f == 0 and se.reshape(g["P"], -1).tolist() == g["base"]
    for M, key in ((1, "microstep_M1"), (2, "microstep_M2")):
        out, f = orc.microstep_placement(c, se, g["P"], g["Nb"], g["Nr"], M)
        assert f == 0 and out.reshape(g["P"], -1).tolist() == g[key]


def test_golden_vector_machines_matter():
    """Second hand-worked vector: micro-step loads that differ from the step totals, so that M = 2
    (relocation / replication confined to each machine) gives another placement than M = 1."""
    g = json.load(open(os.path.join(HERE, "golden", "placement_vectors.json")))
    v = g["second_vector"]
    base, f = orc.base_placement(np.array(v["tot"]), g["P"], g["Nb"], g["Nr"])
    assert f == 0 and base.reshape(g["P"], -1).tolist() == g["base"]
    c = np.array(v["c_mb"], dtype=np.int32)
    outs = {}
    for M in (1, 2):
        out, f = orc.microstep_placement(c, base, g["P"], g["Nb"], g["Nr"], M)
        assert f == 0 and out.reshape(g["P"], -1).tolist() == v[f"microstep_M{M}"], M
        outs[M] = out
        _replay_stage3(c, out, g["P"], g["Nb"], g["Nr"], M)
    assert (outs[1] != outs[2]).any()


def _replay_stage3(c, out, P, Nb, Nr, M):
    """Re-derive every replication round of Alg. 3 Stage 3 (readings 22-25)
    from the OUTPUT alone, independently of the oracle's bookkeeping: the base slots of `out` are the
    Stage-2 result; round by round the expected (expert, rank) is recomputed from scratch -- the locally
    heaviest expert PER COPY (exact fractions, ties lower id) among those that still have an eligible
    rank, on the least-loaded local rank with a free redundant slot that does not host it (ties lowest
    rank), rank loads = sum over experts of the exact integer even split (first c mod n hosts in
    ascending slot index carry one more) -- and must be what `out` holds in that rank's next redundant
    slot.  Slots no round fills must be -1."""
    from fractions import Fraction
    Ns, R, E = Nb + Nr, P // M, len(c)
    se = np.asarray(out).reshape(P, Ns)
    hosts = {e: [] for e in range(E)}                   # global slot indices, base slots first
    for r in range(P):
        for b in range(Nb):
            if se[r, b] >= 0:
                hosts[int(se[r, b])].append(r * Ns + b)
    assert all(len(h) == 1 for h in hosts.values())
    mach = {e: (hosts[e][0] // Ns) // R for e in range(E)}
    filled = [0] * P

    def rank_loads():
        RL = [0] * P
        for e in range(E):
            hs = sorted(hosts[e])
            n = len(hs)
            for idx, j in enumerate(hs):
                RL[j // Ns] += int(c[e]) // n + (1 if idx < int(c[e]) % n else 0)
        return RL

    for m in range(M):
        ranks = range(m * R, (m + 1) * R)
        for _ in range(R * Nr):
            def eligible(e):
                on = {j // Ns for j in hosts[e]}
                return [r for r in ranks if filled[r] < Nr and r not in on]
            cands = [e for e in range(E) if mach[e] == m and c[e] > 0 and eligible(e)]
            if not cands:
                break
            estar = min(cands, key=lambda e: (-Fraction(int(c[e]), len(hosts[e])), e))
            RL = rank_loads()
            rstar = min(eligible(estar), key=lambda r: (RL[r], r))
            assert se[rstar, Nb + filled[rstar]] == estar, (m, estar, rstar, se.tolist())
            hosts[estar].append(rstar * Ns + Nb + filled[rstar])
            filled[rstar] += 1
        for r in ranks:
            assert (se[r, Nb + filled[r]:] == -1).all(), (r, se.tolist())


def test_equal_loads_round_robin():
    E, P, Nb, Nr = 12, 4, 3, 2
    se, f = orc.base_placement(np.full(E, 5), P, Nb, Nr)
    assert f == 0
    exp = np.full((P, Nb + Nr), -1)
    for r in range(P):
        for b in range(Nb):
            exp[r, b] = b * P + r
    assert (se.reshape(P, -1) == exp).all()


def test_one_slot_per_rank_is_sorted_order():
    rng = np.random.default_rng(0)
    c = rng.permutation(16) * 3 + 1
    se, f = orc.base_placement(c, 16, 1, 0)
    assert f == 0 and (se == np.argsort(-c, kind="stable")).all()


def _check_lpt_invariant(c, se, P, Nb, Ns, ranks_of_machine):
    """Replay in (load desc, id asc) order: at its turn every expert sits on a rank whose load was
    minimal among the ranks of its machine that still had a free base slot, lowest rank on ties."""
    order = sorted(range(len(c)), key=lambda e: (-int(c[e]), e))
    where = {int(se[j]): j // Ns for j in range(len(se)) if se[j] >= 0 and j % Ns < Nb}
    RL = np.zeros(P, dtype=np.int64)
    nb = np.zeros(P, dtype=np.int64)
    for e in order:
        r = where[e]
        cand = [q for q in ranks_of_machine(r) if nb[q] < Nb]
        best = min(cand, key=lambda q: (RL[q], q))
        assert r == best, (e, r, best)
        RL[r] += c[e]
        nb[r] += 1
    return RL


@pytest.mark.parametrize("seed", range(8))
def test_random_instances_invariants(seed):
    rng = np.random.default_rng(seed)
    P = int(rng.choice([2, 4, 6, 8]))
    Nb, Nr = int(rng.integers(1, 5)), int(rng.integers(0, 4))
    E, Ns = P * Nb, Nb + Nr
    tot = rng.integers(0, 1000, size=E) * rng.integers(0, 2, size=E)      # some zero loads
    base, f = orc.base_placement(tot, P, Nb, Nr)
    assert f == 0
    _structure_ok(base, E, P, Nb, Nr, base_only=True)
    _check_lpt_invariant(tot, base, P, Nb, Ns, lambda r: range(P))
    c = rng.integers(0, 300, size=E).astype(np.int32) * rng.integers(0, 2, size=E).astype(np.int32)
    for M in [m for m in (1, 2) if P % m == 0]:
        R = P // M
        out, f = orc.microstep_placement(c, base, P, Nb, Nr, M)
        assert f == 0
        _structure_ok(out, E, P, Nb, Nr, c=c)
        _replay_stage3(c, out, P, Nb, Nr, M)              # every replication round, from the output
        RL = _check_lpt_invariant(c, out, P, Nb, Ns, lambda r: range((r // R) * R, (r // R + 1) * R))
        # experts stay on the machine of their base rank; replicas too
        mach = {int(base[j]): (j // Ns) // R for j in range(len(base)) if base[j] >= 0}
        for j, e in enumerate(out):
            if e >= 0:
                assert mach[int(e)] == (j // Ns) // R
        # first replica of each machine: the heaviest local expert, on the least-loaded other rank
        if Nr > 0:
            for m in range(M):
                local = [e for e in range(E) if mach[e] == m and c[e] > 0]
                if not local or R < 2:
                    continue
                e1 = min(local, key=lambda e: (-int(c[e]), e))
                home = [j // Ns for j in range(len(out)) if out[j] == e1 and j % Ns < Nb][0]
                cand = [r for r in range(m * R, (m + 1) * R) if r != home]
                r1 = min(cand, key=lambda r: (RL[r], r))
                assert out[r1 * Ns + Nb] == e1


def test_replication_then_stage4_improves_balance():
    """On a config-3-shaped trace (64 ranks x 1 replica slot is too coarse at step level) the
    per-micro-step Stages 2-3 + Stage 4 bring max/mean rank load down on every instance."""
    cfg = synth.config(3).scaled(L=1, n_samples=8, sample_len=1024, H=64)
    ids, w, mb_off = synth.gen_trace(cfg, "cpu")
    ids, mb_off = ids.numpy(), mb_off.numpy()
    hist, step, f = orc.load_hist(ids, mb_off, cfg.E)
    base, f = orc.base_placement(step[0], cfg.P, cfg.Nb, cfg.Nr)
    assert f == 0
    step_level = synth.gen_placement(cfg, step)[0]
    better = 0
    for i in range(cfg.n_mb):
        _, rl0, _, _, f0 = orc.quota(hist[i, 0], step_level, cfg.P, cfg.Ns)
        se, f1 = orc.microstep_placement(hist[i, 0], base, cfg.P, cfg.Nb, cfg.Nr, 1)
        _, rl1, _, _, f2 = orc.quota(hist[i, 0], se, cfg.P, cfg.Ns)
        assert f0 == 0 and f1 == 0 and f2 == 0
        assert rl1.sum() == rl0.sum()
        better += rl1.max() <= rl0.max()
    assert better == cfg.n_mb


def test_faults():
    c = np.array([3, 2, 1, 1], dtype=np.int32)
    base, f = orc.base_placement(np.array([3, 2, 1, 1]), 2, 2, 1)
    assert f == 0
    bad = base.copy()
    bad[bad == 2] = -1                                   # expert 2 has no base slot
    _, f = orc.microstep_placement(c, bad, 2, 2, 1, 1)
    assert f & orc.FAULT_SLOT_EXPERT
    bad = base.copy()
    bad[0] = 9
    _, f = orc.microstep_placement(c, bad, 2, 2, 1, 1)
    assert f & orc.FAULT_SLOT_EXPERT
    _, f = orc.microstep_placement(np.array([3, -1, 1, 1], dtype=np.int32), base, 2, 2, 1, 1)
    assert f & orc.FAULT_ID_RANGE
    _, f = orc.base_placement(np.array([1, 2, 3]), 1, 2, 0)       # more experts than base slots
    assert f & orc.FAULT_SLOT_EXPERT


# ------------------------------------------------------------------ O13: replication alone
@pytest.mark.parametrize("seed", range(8))
def test_replication_only_composes_with_stage2(seed):
    """O13 on O8's own Stage-2 result (O8 run with N_r = 0, padded) must reproduce O8 in full; and the
    first replica of every machine is the heaviest local expert on the least-loaded other rank."""
    rng = np.random.default_rng(400 + seed)
    P = int(rng.choice([2, 4, 6, 8]))
    Nb, Nr = int(rng.integers(1, 5)), int(rng.integers(1, 4))
    E, Ns = P * Nb, Nb + Nr
    tot = rng.integers(1, 1000, size=E)
    c = (rng.integers(0, 300, size=E) * rng.integers(0, 2, size=E)).astype(np.int32)
    for M in [m for m in (1, 2) if P % m == 0]:
        base, f = orc.base_placement(tot, P, Nb, Nr)
        full, f1 = orc.microstep_placement(c, base, P, Nb, Nr, M)
        base0, _ = orc.base_placement(tot, P, Nb, 0)
        st2, f2 = orc.microstep_placement(c, base0, P, Nb, 0, M)           # Stage 2 only
        padded = np.full(P * Ns, -1, dtype=np.int32)
        padded.reshape(P, Ns)[:, :Nb] = st2.reshape(P, Nb)
        padded.reshape(P, Ns)[:, Nb:] = rng.integers(-1, E, size=(P, Nr))  # garbage: must be ignored
        rep, f3 = orc.replication(c, padded, P, Nb, Nr, M)
        assert f == 0 and f1 == 0 and f2 == 0 and f3 == 0
        assert (rep == full).all()
        _structure_ok(rep, E, P, Nb, Nr, c=c)
        _replay_stage3(c, rep, P, Nb, Nr, M)


@pytest.mark.parametrize("seed", range(12))
def test_replication_only_replay_on_arbitrary_base(seed):
    """O13's own pin (independent of O8): on a RANDOM base placement (any expert on any rank -- what
    Alg. 2's swaps may produce, not an LPT result) every replication round is re-derived from the
    output; base slots come through unchanged and the input's redundant slots are ignored."""
    rng = np.random.default_rng(4400 + seed)
    P = int(rng.choice([2, 3, 4, 6, 8]))
    Nb, Nr = int(rng.integers(1, 5)), int(rng.integers(1, 4))
    E, Ns = P * Nb, Nb + Nr
    c = (rng.integers(0, 50, size=E) * (rng.random(E) < 0.8)).astype(np.int32)
    if seed % 3 == 0:
        c[:] = c[0]                                          # all ties: lower id / lowest rank decide
    placed = np.full((P, Ns), -1, dtype=np.int32)
    placed[:, :Nb] = rng.permutation(E).reshape(P, Nb)
    placed[:, Nb:] = rng.integers(-1, E, size=(P, Nr))       # garbage: must be ignored
    for M in [m for m in (1, 2, P) if P % m == 0]:
        rep, f = orc.replication(c, placed.ravel(), P, Nb, Nr, M)
        assert f == 0
        assert (rep.reshape(P, Ns)[:, :Nb] == placed[:, :Nb]).all()
        _structure_ok(rep, E, P, Nb, Nr, c=c)
        _replay_stage3(c, rep, P, Nb, Nr, M)


def test_replication_only_on_swapped_placement_and_faults():
    c = np.array([9, 8, 1, 2], dtype=np.int32)
    swapped, st, f = orc.swap_relocation(c, np.array([0, 1, -1, 2, 3, -1]), 2, 2, 1, 1, 2, 8)
    assert f == 0 and swapped.tolist() == [3, 1, -1, 2, 0, -1]
    rep, f = orc.replication(c, swapped, 2, 2, 1, 1)
    # rank loads 10 | 10; heaviest per copy e0 (9) -> least-loaded rank not hosting it = rank 0;
    # then e1 (8 vs e0 4.5 per copy) -> rank 1
    assert f == 0 and rep.tolist() == [3, 1, 0, 2, 0, 1]
    bad = swapped.copy(); bad[0] = 1                                       # e1 twice, e3 missing
    rep, f = orc.replication(c, bad, 2, 2, 1, 1)
    assert f & orc.FAULT_SLOT_EXPERT and (rep == -1).all()


# ------------------------------------------------------------------ O14: Alg. 1 in full (machine level + rank level)
def _replay_alg1(tot_me, se, P, Nb, Nr, M, a, b):
    """Re-derive every greedy choice of Alg. 1 from the OUTPUT: at its turn each expert sits on a machine
    of minimal score among those with a free base slot (lowest m on ties), and inside the machine on the
    least-loaded rank with a free base slot."""
    Ns, R = Nb + Nr, P // M
    E = tot_me.shape[1]
    tot = tot_me.sum(0)
    where = {int(se[j]): j // Ns for j in range(len(se)) if se[j] >= 0}
    assert sorted(where) == list(range(E))
    order = sorted(range(E), key=lambda e: (-int(tot[e]), e))
    ML, MC, cnt = np.zeros(M, np.int64), np.zeros(M, np.int64), np.zeros(M, np.int64)
    for e in order:
        m_out = where[e] // R
        scores = {m: a * (ML[m] + tot[e]) + b * (MC[m] + tot[e] - tot_me[m, e]) for m in range(M) if cnt[m] < R * Nb}
        m_best = min(scores, key=lambda m: (scores[m], m))
        assert m_out == m_best, (e, m_out, m_best)
        ML[m_out] += tot[e]; MC[m_out] += tot[e] - tot_me[m_out, e]; cnt[m_out] += 1
    RL, nb = np.zeros(P, np.int64), np.zeros(P, np.int64)
    for e in order:
        r = where[e]
        cand = [q for q in range((r // R) * R, (r // R + 1) * R) if nb[q] < Nb]
        assert r == min(cand, key=lambda q: (RL[q], q))
        RL[r] += tot[e]; nb[r] += 1
    return ML, MC


@pytest.mark.parametrize("seed", range(12))
def test_alg1_machines_replay(seed):
    rng = np.random.default_rng(500 + seed)
    P, M = [(4, 2), (8, 2), (8, 4), (6, 3), (16, 4), (8, 8)][seed % 6]
    Nb, Nr = int(rng.integers(1, 5)), int(rng.integers(0, 3))
    a, b = [(1, 0), (0, 1), (1, 1), (3, 2)][seed % 4]
    E = P * Nb
    tot_me = (rng.integers(0, 1000, size=(M, E)) * (rng.random((M, E)) < 0.7)).astype(np.int64)
    se, f = orc.base_placement_machines(tot_me, P, Nb, Nr, M, a, b)
    assert f == 0
    _structure_ok(se, E, P, Nb, Nr, base_only=True)
    _replay_alg1(tot_me, se, P, Nb, Nr, M, a, b)


def test_alg1_special_cases():
    rng = np.random.default_rng(7)
    # M = 1 is O7
    tot = rng.integers(0, 500, size=24)
    se1, f1 = orc.base_placement_machines(tot.reshape(1, -1), 8, 3, 1, 1, 5, 9)
    se7, f7 = orc.base_placement(tot, 8, 3, 1)
    assert f1 == 0 and f7 == 0 and (se1 == se7).all()
    # a = 0: only inbound traffic counts -> an expert whose tokens all come from one machine lands there
    # (Delta = 0 on that machine, > 0 elsewhere) as long as it has room
    P, M, Nb = 4, 2, 2
    tot_me = np.array([[9, 0, 7, 0, 5, 0, 3, 0], [0, 8, 0, 6, 0, 4, 0, 2]], dtype=np.int64)
    se, f = orc.base_placement_machines(tot_me, P, Nb, 0, M, 0, 1)
    assert f == 0
    mach = {int(e): (j // Nb) // 2 for j, e in enumerate(se)}
    assert all(mach[e] == e % 2 for e in range(8))
    # hand-worked, a = b = 1, M = 2 machines of 1 rank, N_b = 2: loads (m0, m1): e0 (6,0) e1 (1,4) e2 (0,4) e3 (3,0)
    # order e0(6) e1(5) e2(4) e3(3); e0: score m0 = 6+0, m1 = 6+6 -> m0 (ML 6,0; MC 0,0)
    # e1: m0 = (6+5)+(0+4) = 15, m1 = 5+1 = 6 -> m1 (ML 6,5; MC 0,1); e2: m0 = 10+4 = 14, m1 = 9+1+0 = 10 -> m1 (full)
    # e3: only m0 has room -> m0.  ranks = machines: rank0 [e0, e3], rank1 [e1, e2]
    tot_me = np.array([[6, 1, 0, 3], [0, 4, 4, 0]], dtype=np.int64)
    se, f = orc.base_placement_machines(tot_me, 2, 2, 1, 2, 1, 1)
    assert f == 0 and se.tolist() == [0, 3, -1, 1, 2, -1]
    # faults
    bad = tot_me.copy(); bad[0, 0] = -1
    se, f = orc.base_placement_machines(bad, 2, 2, 1, 2, 1, 1)
    assert f & orc.FAULT_ID_RANGE and (se == -1).all()
