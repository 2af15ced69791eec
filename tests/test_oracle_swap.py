"""Pins for oracle O12 (Alg. 2 Stage 2: expert relocation via swaps, listing lines
4-12 :349-372; readings 33-35): hand-worked vectors, the objective recomputed from the placements
with numpy, strict decrease per applied swap, termination = no improving swap in the bottleneck's
window (independent enumeration), structure, brute force over ALL swaps when the window covers the rank."""
import json
import os

import numpy as np
import pytest

from oracle import foremoe_oracle as orc

HERE = os.path.dirname(os.path.abspath(__file__))


def objective(c_me, se, P, Nb, Nr, M, a, b):
    """F = a * L_max + b * C_max from the placement alone (Eq.(3)-(5) with one host per expert)."""
    Ns, R = Nb + Nr, P // M
    c = c_me.sum(0)
    RL = np.zeros(P, dtype=np.int64)
    LT = np.zeros((M, M), dtype=np.int64)
    for j, e in enumerate(se):
        if e >= 0 and j % Ns < Nb:
            RL[j // Ns] += c[e]
            LT[:, (j // Ns) // R] += c_me[:, e]
    np.fill_diagonal(LT, 0)
    return int(a * RL.max() + b * LT.max()), RL


def window_swaps(c_me, se, P, Nb, Nr, win):
    """All swaps Alg. 2 line 6 looks at: (e_h, e_l) with e_h among the `win` heaviest on the bottleneck
    rank and e_l among the `win` lightest on every other rank."""
    Ns = Nb + Nr
    c = c_me.sum(0)
    RL = np.array([sum(int(c[e]) for e in se[r * Ns:r * Ns + Nb] if e >= 0) for r in range(P)])
    h = int(np.argmax(RL))
    on = lambda r: [int(e) for e in se[r * Ns:r * Ns + Nb] if e >= 0]
    heavy = sorted(on(h), key=lambda e: (-int(c[e]), e))[:win]
    out = []
    for r in range(P):
        if r != h:
            light = sorted(on(r), key=lambda e: (int(c[e]), e))[:win]
            out += [(eh, el) for eh in heavy for el in light]
    return out


def swapped(se, eh, el):
    s2 = se.copy()
    jh, jl = int(np.where(se == eh)[0][0]), int(np.where(se == el)[0][0])
    s2[jh], s2[jl] = el, eh
    return s2


def test_golden_vectors():
    g = json.load(open(os.path.join(HERE, "golden", "swap_vectors.json")))
    for v in g["vectors"]:
        out, st, f = orc.swap_relocation(np.array(v["c_me"]), np.array(v["base"]).ravel(), v["P"], v["Nb"],
                                         v["Nr"], v["M"], v["win"], v["max_rounds"], v["a"], v["b"])
        assert f == 0, v["name"]
        assert out.reshape(v["P"], -1).tolist() == v["out"], v["name"]
        assert st.tolist() == [v["rounds"], v["F0"], v["F1"]], v["name"]


def random_case(rng, P, M, Nb, Nr):
    E, Ns = P * Nb, Nb + Nr
    c_me = (rng.integers(0, 300, size=(M, E)) * (rng.random((M, E)) < 0.8)).astype(np.int32)
    base = np.full(P * Ns, -1, dtype=np.int32)
    perm = rng.permutation(E)
    for r in range(P):
        base[r * Ns:r * Ns + Nb] = perm[r * Nb:(r + 1) * Nb]
    return c_me, base


@pytest.mark.parametrize("seed", range(24))
def test_rounds_decrease_and_terminate(seed):
    rng = np.random.default_rng(seed)
    P, M, Nb, Nr = [(4, 1, 4, 1), (8, 2, 4, 2), (8, 8, 2, 0), (6, 3, 5, 1)][seed % 4]
    win = int(rng.integers(1, 4))
    a, b = [(1, 0), (1, 1), (3, 2), (0, 1)][(seed // 4) % 4]
    c_me, base = random_case(rng, P, M, Nb, Nr)
    final, st, f = orc.swap_relocation(c_me, base, P, Nb, Nr, M, win, 64, a, b)
    assert f == 0
    rounds = int(st[0])
    assert rounds < 64
    prev_F, _ = objective(c_me, base, P, Nb, Nr, M, a, b)
    assert prev_F == st[1]
    prev = base
    for r in range(1, rounds + 1):                     # placement after r rounds
        cur, st_r, f = orc.swap_relocation(c_me, base, P, Nb, Nr, M, win, r, a, b)
        F, _ = objective(c_me, cur, P, Nb, Nr, M, a, b)
        assert f == 0 and st_r[0] == r and F == st_r[2] and F < prev_F     # strict decrease
        assert (cur != prev).sum() == 2                                    # exactly one swap per round
        # the applied swap is the best one of the window (first best in enumeration order)
        cands = window_swaps(c_me, prev, P, Nb, Nr, win)
        Fs = [objective(c_me, swapped(prev, eh, el), P, Nb, Nr, M, a, b)[0] for eh, el in cands]
        k = int(np.argmin(Fs))                          # numpy argmin = first minimum
        assert F == Fs[k] and (cur == swapped(prev, *cands[k])).all()
        prev, prev_F = cur, F
    assert (prev == final).all() and prev_F == st[2]
    # termination: no swap of the bottleneck's window improves the objective
    cands = window_swaps(c_me, final, P, Nb, Nr, win)
    assert all(objective(c_me, swapped(final, eh, el), P, Nb, Nr, M, a, b)[0] >= prev_F for eh, el in cands)
    # structure: the base slots hold a permutation of the experts, redundant slots untouched
    Ns = Nb + Nr
    mask = (np.arange(P * Ns) % Ns) < Nb
    assert sorted(final[mask].tolist()) == list(range(P * Nb)) and (final[~mask] == base[~mask]).all()


@pytest.mark.parametrize("seed", range(8))
def test_full_window_two_ranks_is_best_of_all_swaps(seed):
    rng = np.random.default_rng(50 + seed)
    P, M, Nb, Nr = 2, 2, 4, 0
    c_me, base = random_case(rng, P, M, Nb, Nr)
    one, st, f = orc.swap_relocation(c_me, base, P, Nb, Nr, M, Nb, 1, 2, 1)
    F0, _ = objective(c_me, base, P, Nb, Nr, M, 2, 1)
    best = min(objective(c_me, swapped(base, int(eh), int(el)), P, Nb, Nr, M, 2, 1)[0]
               for eh in base[:Nb] for el in base[Nb:])
    assert f == 0 and st[2] == min(F0, best)


def test_balanced_input_unchanged_and_faults():
    c = np.full((1, 8), 5, dtype=np.int32)
    base = np.array([0, 1, -1, 2, 3, -1, 4, 5, -1, 6, 7, -1], dtype=np.int32)
    out, st, f = orc.swap_relocation(c, base, 4, 2, 1, 1, 2, 8)
    assert f == 0 and (out == base).all() and st[0] == 0
    bad = base.copy(); bad[1] = 0                                   # expert 0 twice, expert 1 missing
    out, st, f = orc.swap_relocation(c, bad, 4, 2, 1, 1, 2, 8)
    assert f & orc.FAULT_SLOT_EXPERT and (out == -1).all()
    neg = c.copy(); neg[0, 3] = -1
    out, st, f = orc.swap_relocation(neg, base, 4, 2, 1, 1, 2, 8)
    assert f & orc.FAULT_ID_RANGE
