"""Test-local helpers: tiny random Stage-4 instances and independent re-derivations.

Nothing here is used by the product or by the oracle; these are the *pins* the oracle is held
to (brute force, closed forms, library routines).
"""
from __future__ import annotations

import itertools
import math

import numpy as np


def build_instance(b, experts, extra_dup=False):
    """Placement for Phase-A loads ``b`` (one filler expert per rank) and replicated experts
    ``experts`` = [(count, [ranks...])]; replicated experts get ids 0..n-1 (listed order),
    fillers ids n..n+P-1.  Returns (c[E], slot_expert[S], P, Ns)."""
    P = len(b)
    n = len(experts)
    per_rank = [[] for _ in range(P)]
    for e, (_, ranks) in enumerate(experts):
        for r in ranks:
            per_rank[r].append(e)
    Ns = 1 + max([len(x) for x in per_rank] + [0]) + (1 if extra_dup else 0)
    se = np.full(P * Ns, -1, dtype=np.int32)
    c = np.zeros(n + P, dtype=np.int32)
    for r in range(P):
        se[r * Ns] = n + r
        c[n + r] = b[r]
        for a, e in enumerate(sorted(per_rank[r])):
            se[r * Ns + 1 + a] = e
    for e, (cnt, _) in enumerate(experts):
        c[e] = cnt
    return c, se, P, Ns


def hosts_of(se, Ns, e):
    """Active host slots of e: ascending slot index, only the first slot per rank."""
    out, seen = [], set()
    for j, v in enumerate(se):
        if v == e and (j // Ns) not in seen:
            seen.add(j // Ns)
            out.append(j)
    return out


def compositions(total, parts):
    """All ways to write ``total`` as an ordered sum of ``parts`` non-negative integers."""
    if parts == 1:
        yield (total,)
        return
    for first in range(total + 1):
        for rest in compositions(total - first, parts - 1):
            yield (first,) + rest


def brute_force_min_max_load(c, se, P, Ns):
    """Minimum over ALL integer splits of every replicated expert of the maximum rank load."""
    E = len(c)
    base = np.zeros(P, dtype=np.int64)
    rep = []
    for e in range(E):
        h = hosts_of(se, Ns, e)
        if len(h) == 1:
            base[h[0] // Ns] += c[e]
        elif len(h) >= 2:
            rep.append((e, [j // Ns for j in h]))
        else:
            assert c[e] == 0
    best = None
    choices = [list(compositions(int(c[e]), len(rk))) for e, rk in rep]
    for combo in itertools.product(*choices):
        load = base.copy()
        for (e, rk), split in zip(rep, combo):
            for r, s in zip(rk, split):
                load[r] += s
        m = int(load.max())
        if best is None or m < best:
            best = m
    return best


def subset_closed_form(c, se, P, Ns):
    """max over non-empty A of ceil((sum_{r in A} b_r + sum_{e in R, hosts(e) in A} c_e)/|A|):
    the Hall-type lower bound that an optimal assignment attains."""
    E = len(c)
    base = np.zeros(P, dtype=np.int64)
    rep = []
    for e in range(E):
        h = hosts_of(se, Ns, e)
        if len(h) == 1:
            base[h[0] // Ns] += c[e]
        elif len(h) >= 2:
            rep.append((int(c[e]), frozenset(j // Ns for j in h)))
    best = 0
    for mask in range(1, 1 << P):
        A = frozenset(r for r in range(P) if mask >> r & 1)
        tot = sum(int(base[r]) for r in A) + sum(cnt for cnt, rk in rep if rk <= A)
        best = max(best, -(-tot // len(A)))
    return best


def lp_min_max_load(c, se, P, Ns):
    """LP Eq.(10) of the paper with one machine (C* dropped): minimise L* subject to
    conservation and feasibility, solved by HiGHS through scipy (the paper's solver family,
    PAPER.md:407).  Returns the LP optimum (float)."""
    from scipy.optimize import linprog
    E = len(c)
    base = np.zeros(P)
    var = []          # (expert, rank)
    for e in range(E):
        h = hosts_of(se, Ns, e)
        if len(h) == 1:
            base[h[0] // Ns] += c[e]
        elif len(h) >= 2:
            for j in h:
                var.append((e, j // Ns))
    if not var:
        return float(base.max())
    nv = len(var)
    cost = np.zeros(nv + 1)
    cost[nv] = 1.0
    reps = sorted(set(e for e, _ in var))
    A_eq = np.zeros((len(reps), nv + 1))
    b_eq = np.zeros(len(reps))
    for row, e in enumerate(reps):
        for v, (e2, _) in enumerate(var):
            if e2 == e:
                A_eq[row, v] = 1.0
        b_eq[row] = c[e]
    A_ub = np.zeros((P, nv + 1))
    b_ub = -base.copy()
    for v, (_, r) in enumerate(var):
        A_ub[r, v] = 1.0
    A_ub[:, nv] = -1.0
    res = linprog(cost, A_ub=A_ub, b_ub=b_ub, A_eq=A_eq, b_eq=b_eq,
                  bounds=[(0, None)] * (nv + 1), method="highs")
    assert res.status == 0, res.message
    return float(res.fun)


def random_tiny_instance(rng, max_P=5, max_rep=4, max_cnt=12, max_hosts=3, combos_cap=20000):
    while True:
        P = int(rng.integers(2, max_P + 1))
        n = int(rng.integers(1, max_rep + 1))
        b = [int(x) for x in rng.integers(0, max_cnt + 1, size=P)]
        experts = []
        combos = 1
        for _ in range(n):
            h = int(rng.integers(2, min(P, max_hosts) + 1))
            ranks = sorted(int(x) for x in rng.choice(P, size=h, replace=False))
            cnt = int(rng.integers(0, max_cnt + 1))
            combos *= math.comb(cnt + h - 1, h - 1)
            experts.append((cnt, ranks))
        if combos <= combos_cap:
            return b, experts
