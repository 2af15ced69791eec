"""Pins for oracle O11 (locality-aware, per-source Stage 4 over M machines):
PAPER.md:337 (prefer same-machine replicas, leftover tokens minimise per-rank load), Eq.(4)/(5)
:254-258, Eq.(10) :397-405.  Brute force, the restricted LP (HiGHS), the traffic lower bound, the
M = 1 and single-machine special cases, hand-worked vectors."""
import itertools
import json
import math
import os

import numpy as np
import pytest

from oracle import foremoe_oracle as orc
from tests import helpers as Hh

HERE = os.path.dirname(os.path.abspath(__file__))


def allowed_hosts(se, Ns, R, e, m):
    """Re-derivation of the rule in Python: active hosts (first slot per rank) of e on machine m if
    the machine holds e, else all active hosts."""
    h = Hh.hosts_of(se, Ns, e)
    local = [j for j in h if (j // Ns) // R == m]
    return local if local else h


def commodities(w_se, se, P, Ns, M):
    R = P // M
    E = w_se.shape[1]
    out = []
    for e in range(E):
        for m in range(M):
            cnt = int(w_se[m * R:(m + 1) * R, e].sum())
            if cnt:
                out.append((e, m, cnt, allowed_hosts(se, Ns, R, e, m)))
    return out


def brute_force(w_se, se, P, Ns, M):
    com = commodities(w_se, se, P, Ns, M)
    choices = [list(Hh.compositions(cnt, len(h))) for (_, _, cnt, h) in com]
    best = None
    for combo in itertools.product(*choices):
        load = np.zeros(P, dtype=np.int64)
        for (_, _, _, h), split in zip(com, combo):
            for j, s in zip(h, split):
                load[j // Ns] += s
        best = int(load.max()) if best is None else min(best, int(load.max()))
    return best


def lp_restricted(w_se, se, P, Ns, M):
    """Eq.(10) with r_{s,e,j} forced to 0 outside the allowed hosts and the C* term dropped (the
    restriction already makes every C_{i,j} minimal): minimise L*."""
    from scipy.optimize import linprog
    com = commodities(w_se, se, P, Ns, M)
    var = [(ci, j // Ns) for ci, (_, _, _, h) in enumerate(com) for j in h]
    nv = len(var)
    cost = np.zeros(nv + 1)
    cost[nv] = 1.0
    A_eq = np.zeros((len(com), nv + 1))
    b_eq = np.array([c[2] for c in com], dtype=float)
    A_ub = np.zeros((P, nv + 1))
    for v, (ci, r) in enumerate(var):
        A_eq[ci, v] = 1.0
        A_ub[r, v] = 1.0
    A_ub[:, nv] = -1.0
    res = linprog(cost, A_ub=A_ub, b_ub=np.zeros(P), A_eq=A_eq, b_eq=b_eq,
                  bounds=[(0, None)] * (nv + 1), method="highs")
    assert res.status == 0, res.message
    return float(res.fun)


def random_instance(rng, P, M, Nb, Nr, max_cnt, p_rep=0.7):
    """Random placement: every expert once in a base slot, replicas anywhere (other ranks)."""
    Ns, E = Nb + Nr, P * Nb
    se = np.full(P * Ns, -1, dtype=np.int32)
    perm = rng.permutation(E)
    for r in range(P):
        se[r * Ns:r * Ns + Nb] = perm[r * Nb:(r + 1) * Nb]
        for a in range(Nr):
            if rng.random() < p_rep:
                se[r * Ns + Nb + a] = int(rng.integers(0, E))      # may duplicate an expert of the rank
    w_se = (rng.integers(0, max_cnt + 1, size=(P, E)) * (rng.random((P, E)) < 0.6)).astype(np.int32)
    return w_se, se, Ns, E


def check_invariants(w_se, se, P, Ns, M, out):
    R = P // M
    E = w_se.shape[1]
    S = P * Ns
    q = out["q_src"]
    assert out["fault"] == 0 and (q >= 0).all()
    for e in range(E):
        for m in range(M):
            cnt = int(w_se[m * R:(m + 1) * R, e].sum())
            ok = allowed_hosts(se, Ns, R, e, m)
            got = {j: int(q[m, j]) for j in range(S) if se[j] == e and q[m, j]}
            assert sum(got.values()) == cnt                       # Eq.(8) per (source machine, expert)
            assert set(got) <= set(ok)                            # Eq.(9) + the locality rule
    assert (q[:, se < 0] == 0).all()
    assert (out["rank_load"] == q.sum(0).reshape(P, Ns).sum(1)).all()          # Eq.(4)
    tr = q.reshape(M, M, R * Ns).sum(-1)
    assert (out["traffic"] == tr).all()                                        # Eq.(5)
    # total cross-machine traffic = its lower bound: the tokens whose expert has no local replica
    forced = 0
    for e in range(E):
        hosts_m = {(j // Ns) // R for j in range(S) if se[j] == e}
        for m in range(M):
            if m not in hosts_m:
                forced += int(w_se[m * R:(m + 1) * R, e].sum())
    assert int(tr.sum() - np.trace(tr)) == forced
    assert (out["quota_v"].reshape(S, M).T == q).all()
    assert (out["slot_off_v"] == np.concatenate([[0], np.cumsum(out["quota_v"])])).all()


def test_golden_vectors():
    g = json.load(open(os.path.join(HERE, "golden", "local_vectors.json")))
    for v in g["vectors"]:
        w = np.array(v["w_se"], dtype=np.int32)
        out = orc.quota_local(w, np.array(v["slot_expert"]), v["P"], v["Ns"], v["M"])
        assert out["fault"] == 0, v["name"]
        assert out["q_src"].tolist() == v["q_src"], v["name"]
        assert out["rank_load"].tolist() == v["rank_load"], v["name"]
        assert out["traffic"].tolist() == v["traffic"], v["name"]


@pytest.mark.parametrize("seed", range(40))
def test_brute_force_optimum_tiny(seed):
    rng = np.random.default_rng(seed)
    while True:
        P, M = [(2, 2), (4, 2), (3, 1), (4, 4), (6, 3), (6, 2)][seed % 6]
        w_se, se, Ns, E = random_instance(rng, P, M, Nb=1, Nr=int(rng.integers(1, 3)), max_cnt=5)
        com = commodities(w_se, se, P, Ns, M)
        combos = math.prod(math.comb(c[2] + len(c[3]) - 1, len(c[3]) - 1) for c in com)
        if combos <= 30000:
            break
    out = orc.quota_local(w_se, se, P, Ns, M)
    check_invariants(w_se, se, P, Ns, M, out)
    assert int(out["rank_load"].max()) == brute_force(w_se, se, P, Ns, M)


@pytest.mark.parametrize("seed", range(12))
def test_restricted_lp_config_shaped(seed):
    rng = np.random.default_rng(100 + seed)
    P, M, Nb, Nr = [(8, 2, 16, 2), (16, 4, 8, 2), (32, 4, 4, 1), (8, 8, 4, 3)][seed % 4]
    w_se, se, Ns, E = random_instance(rng, P, M, Nb, Nr, max_cnt=400, p_rep=0.9)
    out = orc.quota_local(w_se, se, P, Ns, M)
    check_invariants(w_se, se, P, Ns, M, out)
    lp = lp_restricted(w_se, se, P, Ns, M)
    assert int(out["rank_load"].max()) == math.ceil(lp - 1e-7)


@pytest.mark.parametrize("seed", range(6))
def test_one_machine_is_O2(seed):
    rng = np.random.default_rng(200 + seed)
    P, Nb, Nr = 8, 4, 2
    w_se, se, Ns, E = random_instance(rng, P, 1, Nb, Nr, max_cnt=300)
    out = orc.quota_local(w_se, se, P, Ns, 1)
    q, rl, so, _, f = orc.quota(w_se.sum(0).astype(np.int32), se, P, Ns)
    assert f == 0 and (out["q_src"][0] == q).all() and (out["rank_load"] == rl).all()
    assert out["traffic"].tolist() == [[int(w_se.sum())]]


@pytest.mark.parametrize("seed", range(6))
def test_intra_machine_replicas_only(seed):
    """The Alg. 3 setting: every expert's replicas sit on its home machine, so the
    source does not restrict anything and cross traffic is fixed: same optimum as O2 on the sums."""
    rng = np.random.default_rng(300 + seed)
    P, M, Nb, Nr = 8, 2, 4, 2
    R, Ns, E = P // M, Nb + Nr, P * Nb
    se = np.full(P * Ns, -1, dtype=np.int32)
    perm = rng.permutation(E)
    home = {}
    for r in range(P):
        se[r * Ns:r * Ns + Nb] = perm[r * Nb:(r + 1) * Nb]
        for e in perm[r * Nb:(r + 1) * Nb]:
            home[int(e)] = r // R
    for r in range(P):
        local = [e for e, m in home.items() if m == r // R]
        se[r * Ns + Nb:r * Ns + Ns] = rng.choice(local, size=Nr, replace=False)
    w_se = rng.integers(0, 200, size=(P, E)).astype(np.int32)
    out = orc.quota_local(w_se, se, P, Ns, M)
    check_invariants(w_se, se, P, Ns, M, out)
    _, rl, _, _, f = orc.quota(w_se.sum(0).astype(np.int32), se, P, Ns)
    assert f == 0 and int(out["rank_load"].max()) == int(rl.max())
    # cross traffic C_{i,j} = tokens of machine i's sources for experts homed on machine j
    for i in range(M):
        for j in range(M):
            exp = sum(int(w_se[i * R:(i + 1) * R, e].sum()) for e, m in home.items() if m == j)
            assert int(out["traffic"][i, j]) == exp


def test_faults():
    out = orc.quota_local(np.array([[1, 1], [0, 0]]), np.array([0, -1, 0, -1]), 2, 2, 2)
    assert out["fault"] & orc.FAULT_NO_HOST                      # e1 has tokens and no slot
    out = orc.quota_local(np.array([[1, 1], [0, 0]]), np.array([0, 5, 1, -1]), 2, 2, 2)
    assert out["fault"] & orc.FAULT_SLOT_EXPERT
