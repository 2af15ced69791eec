"""Pins for oracle O15 (per-source Stage 4 under F = a * L_max + b * C_max, Eq.(10) PAPER.md:397-405,
as a ladder of locality thresholds; reading 39).  The ends of the ladder are pinned to
O11 and O2, the selection to a numpy recomputation, the value to the LP of Eq.(10) INCLUDING the
C rows (HiGHS) from below and to the integer brute force on tiny instances; one hand-worked vector."""
import itertools
import json
import math
import os

import numpy as np
import pytest

from oracle import foremoe_oracle as orc
from tests import helpers as Hh
from tests.test_oracle_local import random_instance

HERE = os.path.dirname(os.path.abspath(__file__))
LADDER = orc.DEFAULT_LADDER


def _members(w_se, se, P, Ns, M):
    """Every ladder member recomputed step by step through the pinned O2: (L_max, C_max, quota_v, se_v)."""
    R, E, S = P // M, w_se.shape[1], P * Ns
    c_v = w_se.reshape(M, R, E).sum(1).T.reshape(-1).astype(np.int32)          # [E*M], v = e*M + m
    total = int(c_v.sum())
    out = []
    for (num, den) in LADDER:
        # the rule, re-derived in Python
        se_v = np.full(S * M, -1, dtype=np.int32)
        for e in range(E):
            ranks = sorted({j // Ns for j in range(S) if se[j] == e})
            for m in range(M):
                n_loc = sum(1 for r in ranks if r // R == m)
                spill = n_loc > 0 and den > 0 and int(c_v[e * M + m]) * den * P > num * n_loc * total
                for j in range(S):
                    if se[j] == e and ((j // Ns) // R == m or n_loc == 0 or spill):
                        se_v[j * M + m] = e * M + m
        got, f = orc.local_placement_theta(c_v, se, E, P, Ns, M, num, den)
        assert f == 0 and (got == se_v).all(), (num, den)
        q, rl, so, _, f = orc.quota(c_v, se_v, P, Ns * M)
        assert f == 0
        tr = q.reshape(S, M).T.reshape(M, M, R * Ns).sum(-1)                    # [src machine][dst machine]
        off = tr.copy()
        np.fill_diagonal(off, 0)
        out.append((int(rl.max()), int(off.max()) if M > 1 else 0, q, se_v, rl, tr))
    return out


@pytest.mark.parametrize("seed", range(16))
def test_members_selection_and_ends(seed):
    rng = np.random.default_rng(7000 + seed)
    P, M, Nb, Nr = [(8, 2, 4, 2), (8, 4, 2, 2), (16, 4, 4, 1), (6, 3, 2, 2)][seed % 4]
    a, b = [(1, 0), (1, 1), (1, 4), (3, 1), (0, 1), (2, 7)][seed % 6]
    w_se, se, Ns, E = random_instance(rng, P, M, Nb, Nr, max_cnt=60, p_rep=0.9)
    w_se[:P // M] *= 3                                   # machine 0's sources are heavier: locality costs load
    out = orc.quota_tradeoff(w_se, se, P, Ns, M, a, b)
    assert out["fault"] == 0
    mem = _members(w_se, se, P, Ns, M)
    F = [a * lm + b * cm for (lm, cm, *_rest) in mem]
    assert out["F"].tolist() == F
    k = int(np.argmin(F))                                # numpy: first minimum = earliest member
    assert out["member"] == k
    lm, cm, q, se_v, rl, tr = mem[k]
    assert (out["quota_v"] == q).all() and (out["se_v"] == se_v).all()
    assert (out["rank_load"] == rl).all() and (out["traffic"] == tr).all()
    assert (out["q_src"] == q.reshape(P * Ns, M).T).all()
    assert (out["slot_off_v"] == np.concatenate([[0], np.cumsum(q)])).all()
    # ends of the ladder: theta = infinity is O11, theta = 0 reaches O2's optimum on the summed counts
    hard = orc.quota_local(w_se, se, P, Ns, M)
    assert (mem[0][2] == hard["quota_v"]).all()
    _, rl0, _, _, f = orc.quota(w_se.sum(0).astype(np.int32), se, P, Ns)
    assert f == 0 and mem[-1][0] == int(rl0.max())
    # a descending ladder only ever widens the allowed hosts: L_max is non-increasing along it
    lmaxes = [m_[0] for m_ in mem]
    assert all(x >= y for x, y in zip(lmaxes, lmaxes[1:]))
    # never worse than either end
    assert min(F) <= F[0] and min(F) <= F[-1]


def _lp_eq10(w_se, se, P, Ns, M, a, b):
    """Eq.(10) as printed: min a L* + b C*, every copy of e allowed for every source machine."""
    from scipy.optimize import linprog
    R, E, S = P // M, w_se.shape[1], P * Ns
    com = [(e, m, int(w_se[m * R:(m + 1) * R, e].sum())) for e in range(E) for m in range(M)]
    com = [c for c in com if c[2] > 0]
    hosts = {e: Hh.hosts_of(se, Ns, e) for e in range(E)}
    var = [(ci, j) for ci, (e, m, _) in enumerate(com) for j in hosts[e]]
    nv = len(var)
    cost = np.zeros(nv + 2)
    cost[nv], cost[nv + 1] = a, b
    A_eq = np.zeros((len(com), nv + 2))
    b_eq = np.array([c[2] for c in com], dtype=float)
    A_ub = np.zeros((P + M * M, nv + 2))
    for v, (ci, j) in enumerate(var):
        A_eq[ci, v] = 1.0
        A_ub[j // Ns, v] = 1.0
        mi, mj = com[ci][1], (j // Ns) // R
        if mi != mj:
            A_ub[P + mi * M + mj, v] = 1.0
    A_ub[:P, nv] = -1.0
    A_ub[P:, nv + 1] = -1.0
    res = linprog(cost, A_ub=A_ub, b_ub=np.zeros(P + M * M), A_eq=A_eq, b_eq=b_eq,
                  bounds=[(0, None)] * (nv + 2), method="highs")
    assert res.status == 0, res.message
    return float(res.fun)


@pytest.mark.parametrize("seed", range(10))
def test_lp_of_eq10_is_a_lower_bound(seed):
    rng = np.random.default_rng(7100 + seed)
    P, M, Nb, Nr = [(8, 2, 8, 2), (16, 4, 4, 2), (8, 4, 4, 2)][seed % 3]
    a, b = [(1, 1), (1, 3), (2, 1), (1, 0), (0, 1)][seed % 5]
    w_se, se, Ns, E = random_instance(rng, P, M, Nb, Nr, max_cnt=300, p_rep=0.9)
    out = orc.quota_tradeoff(w_se, se, P, Ns, M, a, b)
    assert out["fault"] == 0
    lp = _lp_eq10(w_se, se, P, Ns, M, a, b)
    F = int(out["F"][out["member"]])
    assert F >= lp - 1e-6                                 # any integer assignment is LP-feasible
    if b == 0:
        assert F == a * math.ceil(lp / a - 1e-7)          # pure load balancing: the exact optimum (member theta = 0)


def _brute_force_F(w_se, se, P, Ns, M, a, b):
    R, E = P // M, w_se.shape[1]
    com = [(e, m, int(w_se[m * R:(m + 1) * R, e].sum()), Hh.hosts_of(se, Ns, e)) for e in range(E) for m in range(M)]
    com = [c for c in com if c[2] > 0]
    choices = [list(Hh.compositions(c[2], len(c[3]))) for c in com]
    best = None
    for combo in itertools.product(*choices):
        load = np.zeros(P, dtype=np.int64)
        tr = np.zeros((M, M), dtype=np.int64)
        for (e, m, _, h), split in zip(com, combo):
            for j, s in zip(h, split):
                load[j // Ns] += s
                tr[m, (j // Ns) // R] += s
        np.fill_diagonal(tr, 0)
        f = a * int(load.max()) + b * int(tr.max())
        best = f if best is None else min(best, f)
    return best


@pytest.mark.parametrize("seed", range(24))
def test_brute_force_tiny(seed):
    """Integer optimum of Eq.(10) by enumeration: a lower bound for the ladder (which restricts the
    allowed hosts), reached exactly whenever b = 0; the rate at which it is reached otherwise is
    reported by test_brute_force_hit_rate."""
    rng = np.random.default_rng(7200 + seed)
    a, b = [(1, 0), (1, 1), (1, 2), (2, 1)][seed % 4]
    while True:
        P, M = [(2, 2), (4, 2), (4, 4)][seed % 3]
        w_se, se, Ns, E = random_instance(rng, P, M, Nb=1, Nr=int(rng.integers(1, 3)), max_cnt=4)
        R = P // M
        combos = 1
        for e in range(E):
            h = len(Hh.hosts_of(se, Ns, e))
            for m in range(M):
                c = int(w_se[m * R:(m + 1) * R, e].sum())
                if c:
                    combos *= math.comb(c + h - 1, h - 1)
        if combos <= 20000:
            break
    out = orc.quota_tradeoff(w_se, se, P, Ns, M, a, b)
    opt = _brute_force_F(w_se, se, P, Ns, M, a, b)
    F = int(out["F"][out["member"]])
    assert F >= opt
    if b == 0:
        assert F == opt


def test_golden_vector():
    g = json.load(open(os.path.join(HERE, "golden", "tradeoff_vectors.json")))
    for v in g["vectors"]:
        w = np.array(v["w_se"], dtype=np.int32)
        for case in v["cases"]:
            out = orc.quota_tradeoff(w, np.array(v["slot_expert"]), v["P"], v["Ns"], v["M"], case["a"], case["b"])
            assert out["fault"] == 0
            assert out["F"].tolist() == case["F"], (v["name"], case)
            assert out["member"] == case["member"], (v["name"], case)
            assert out["rank_load"].tolist() == case["rank_load"]
            assert out["traffic"].tolist() == case["traffic"]
