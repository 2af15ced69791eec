"""Pins for oracle O16 (Alg. 2 Stage 3, replica search, listing :374-378; DESIGN.md
reading 40).  The paper prints no example and no implementation exists, so the oracle is held to an
INDEPENDENT replay: every round is re-derived from the output by a Python implementation that uses the
closed-form water-fill (sort + level) where the oracle assigns token by token, rebuilds the candidate
set from the placement, and recomputes F from its own flows."""
import json
import os

import numpy as np
import pytest

from oracle import foremoe_oracle as orc

HERE = os.path.dirname(os.path.abspath(__file__))


def water_fill(hosts, c):
    """hosts: [(rank, load)]; c tokens, each to the least-loaded host, ties lowest rank -- closed form:
    level lam = largest integer with sum max(0, lam - load) <= c; the remainder goes one each to the
    hosts with load <= lam in ascending rank.  Returns {rank: tokens}."""
    if c == 0:
        return {r: 0 for r, _ in hosts}
    loads = sorted(l for _, l in hosts)
    lo, hi = loads[0], loads[0] + c
    while lo < hi:                                    # largest lam with need(lam) <= c
        mid = (lo + hi + 1) // 2
        if sum(max(0, mid - l) for l in loads) <= c:
            lo = mid
        else:
            hi = mid - 1
    lam = lo
    give = {r: max(0, lam - l) for r, l in hosts}
    rem = c - sum(give.values())
    for r, l in sorted(hosts):
        if rem and l <= lam:
            give[r] += 1
            rem -= 1
    assert rem == 0
    return give


class Replay:
    def __init__(self, c_me, placed, P, Nb, Nr, M, a, b, max_copies):
        self.c, self.P, self.Nb, self.Nr, self.M, self.a, self.b, self.maxc = c_me, P, Nb, Nr, M, a, b, max_copies
        self.Ns, self.R, self.E = Nb + Nr, P // M, c_me.shape[1]
        self.hosts = {e: [] for e in range(self.E)}           # ranks
        self.flow = {}                                        # (e, rank) -> [M]
        placed = np.asarray(placed).reshape(P, self.Ns)
        for r in range(P):
            for e in placed[r, :Nb]:
                if e >= 0:
                    self.hosts[int(e)].append(r)
                    self.flow[(int(e), r)] = [int(c_me[m, e]) for m in range(M)]
        self.filled = [0] * P

    def loads(self, flow=None):
        flow = self.flow if flow is None else flow
        RL = [0] * self.P
        LT = np.zeros((self.M, self.M), dtype=np.int64)
        for (e, r), f in flow.items():
            RL[r] += sum(f)
            for m in range(self.M):
                LT[m, r // self.R] += f[m]
        return RL, LT

    def F(self, flow=None):
        RL, LT = self.loads(flow)
        off = LT.copy()
        np.fill_diagonal(off, 0)
        return self.a * max(RL) + self.b * (int(off.max()) if self.M > 1 else 0)

    def estimate(self, e, r_new):
        flow = {k: v for k, v in self.flow.items() if k[0] != e}
        RL, _ = self.loads(flow)
        hosts = sorted(self.hosts[e] + [r_new])
        new = {r: [0] * self.M for r in hosts}
        for m in sorted(range(self.M), key=lambda m: (-int(self.c[m, e]), m)):
            cnt = int(self.c[m, e])
            if cnt == 0:
                continue
            local = [r for r in hosts if r // self.R == m]
            allowed = local if local else hosts
            give = water_fill([(r, RL[r]) for r in allowed], cnt)
            for r, g in give.items():
                RL[r] += g
                new[r][m] += g
        for r in hosts:
            flow[(e, r)] = new[r]
        return flow

    def best(self):
        F0 = self.F()
        best = None
        for e in range(self.E):
            if self.c[:, e].sum() <= 0 or len(self.hosts[e]) >= self.maxc:
                continue
            for r in range(self.P):
                if self.filled[r] >= self.Nr or r in self.hosts[e]:
                    continue
                flow = self.estimate(e, r)
                d = self.F(flow) - F0
                if d < 0 and (best is None or d < best[0]):
                    best = (d, e, r, flow)
        return best

    def run_against(self, out):
        out = np.asarray(out).reshape(self.P, self.Ns)
        rounds = 0
        Fs = [self.F()]
        for _ in range(self.P * self.Nr):
            b = self.best()
            if b is None:
                break
            d, e, r, flow = b
            assert out[r, self.Nb + self.filled[r]] == e, (rounds, e, r, out.tolist())
            self.flow = flow
            self.hosts[e].append(r)
            self.filled[r] += 1
            rounds += 1
            Fs.append(self.F())
        for r in range(self.P):
            assert (out[r, self.Nb + self.filled[r]:] == -1).all(), (r, out.tolist())
        return rounds, Fs


def _random(rng, P, M, Nb, Nr, max_cnt=60, skew=True):
    E = P * Nb
    placed = np.full((P, Nb + Nr), -1, dtype=np.int32)
    placed[:, :Nb] = rng.permutation(E).reshape(P, Nb)
    placed[:, Nb:] = rng.integers(-1, E, size=(P, Nr))          # garbage: not read
    c = (rng.integers(0, max_cnt, size=(M, E)) * (rng.random((M, E)) < 0.7)).astype(np.int32)
    if skew:
        hot = rng.choice(E, size=max(1, E // 6), replace=False)
        c[:, hot] *= 6
    return c, placed.ravel()


@pytest.mark.parametrize("seed", range(24))
def test_every_round_replayed(seed):
    rng = np.random.default_rng(8000 + seed)
    P, M = [(4, 1), (4, 2), (8, 2), (8, 4), (6, 3), (8, 8)][seed % 6]
    Nb, Nr = int(rng.integers(1, 4)), int(rng.integers(1, 3))
    a, b = [(1, 0), (1, 1), (2, 1), (1, 3)][seed % 4]
    maxc = [8, 2, 3][seed % 3]
    c, placed = _random(rng, P, M, Nb, Nr)
    out, stats, f = orc.replica_search(c, placed, P, Nb, Nr, M, a, b, max_copies=maxc)
    assert f == 0
    Ns = Nb + Nr
    assert (out.reshape(P, Ns)[:, :Nb] == placed.reshape(P, Ns)[:, :Nb]).all()       # base slots untouched
    for r in range(P):                                                              # never twice on a rank
        live = out.reshape(P, Ns)[r]
        live = live[live >= 0]
        assert len(set(live.tolist())) == len(live)
    assert np.bincount(out[out >= 0], minlength=P * Nb).max() <= maxc
    rp = Replay(c, placed, P, Nb, Nr, M, a, b, maxc)
    rounds, Fs = rp.run_against(out)
    assert rounds == int(stats[0]) and Fs[0] == int(stats[1]) and Fs[-1] == int(stats[2])
    assert all(x > y for x, y in zip(Fs, Fs[1:]))                                    # every replica pays


def test_hot_expert_is_replicated_until_it_stops_paying():
    """One hot expert (100 tokens) among cold ones (1 each), M = 1, b = 0: the replicas go to the least
    loaded ranks in turn and stop when max load cannot drop (closed form: level of the water-fill)."""
    P, Nb, Nr = 4, 2, 1
    c = np.array([[100, 1, 1, 1, 1, 1, 1, 1]], dtype=np.int32)
    placed = np.array([0, 1, -1, 2, 3, -1, 4, 5, -1, 6, 7, -1])
    out, stats, f = orc.replica_search(c, placed, P, Nb, Nr, 1, 1, 0)
    assert f == 0
    # round 1: loads [101,2,2,2] -> e0 on r1: 100 tokens over r0 (other 1) and r1 (2): 51/50 -> F 52;
    # round 2: -> r2: 103 tokens + ... level: (1 + 2 + 2 + 100) / 3 = 35 -> F 35; round 3: -> r3: (107)/4 -> 27
    assert out.reshape(4, 3)[:, 2].tolist() == [-1, 0, 0, 0]
    assert stats.tolist() == [3, 101, 27]


def test_locality_decides_between_equal_load_candidates():
    """Two machines, b > 0: a replica on the machine whose sources send the tokens removes cross traffic,
    a replica elsewhere does not; both balance the load equally."""
    P, Nb, Nr, M = 4, 1, 1, 2
    # e0 lives on r0 (machine 0) but all its tokens come from machine 1's sources
    c = np.array([[0, 2, 2, 2], [40, 0, 0, 0]], dtype=np.int32)
    placed = np.array([0, -1, 1, -1, 2, -1, 3, -1])
    out, stats, f = orc.replica_search(c, placed, P, Nb, Nr, M, 1, 1)
    assert f == 0
    # F0 = 40 + 40.  Candidate (e0, r2) [machine 1]: commodity (e0, m1) now has a local copy -> all 40
    # tokens on r2 (hard preference): loads [0,2,42,2], cross 0 -> F = 42 + max(LT offdiag) = 42 + 2.
    # Candidate (e0, r1) [machine 0]: no local copy for m1 -> split over r0, r1: 21/19: F = 21 + 40.
    assert out.reshape(4, 2)[:, 1].tolist()[2] == 0 and int(stats[1]) == 80
    rp = Replay(c, placed, P, Nb, Nr, M, 1, 1, 8)
    rp.run_against(out)


def test_golden_vector():
    g = json.load(open(os.path.join(HERE, "golden", "replica_search_vectors.json")))
    for v in g["vectors"]:
        c = np.array(v["c_me"], dtype=np.int32)
        out, stats, f = orc.replica_search(c, np.array(v["placed"]), v["P"], v["Nb"], v["Nr"], v["M"], v["a"], v["b"],
                                           max_copies=v["max_copies"])
        assert f == 0
        assert out.reshape(v["P"], -1).tolist() == v["out"], v["name"]
        assert stats.tolist() == v["stats"], v["name"]


def test_faults():
    c = np.array([[3, 2, 1, 1]], dtype=np.int32)
    out, _, f = orc.replica_search(c, np.array([0, 1, -1, 2, 2, -1]), 2, 2, 1)         # e2 twice, e3 missing
    assert f & orc.FAULT_SLOT_EXPERT and (out == -1).all()
    out, _, f = orc.replica_search(c, np.array([0, 1, -1, 2, 9, -1]), 2, 2, 1)
    assert f & orc.FAULT_SLOT_EXPERT
    out, _, f = orc.replica_search(np.array([[3, -2, 1, 1]], dtype=np.int32), np.array([0, 1, -1, 2, 3, -1]), 2, 2, 1)
    assert f & orc.FAULT_ID_RANGE and (out == -1).all()
