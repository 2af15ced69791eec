"""ctypes + numpy front end of oracle/foremoe_oracle.c -- TEST INFRASTRUCTURE ONLY.

Argument marshalling only; every step is computed by the plain C in foremoe_oracle.c (see its
header for the citations and the pins).  All arrays are host numpy arrays.  bf16 rows are
carried as uint16 bit patterns.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np

from . import build as _build

FAULT_ID_RANGE = 1
FAULT_NO_HOST = 2
FAULT_SLOT_EXPERT = 4
FAULT_MB_OFF = 8
FAULT_QUOTA_IN = 16

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def load_hist(ids: np.ndarray, mb_off: np.ndarray, E: int, want_step: bool = True):
    """O1.  ids int32 [L,T,K] -> hist int32 [n_mb,L,E], step_hist int64 [L,E], fault bits."""
    ids = _i32(ids)
    mb_off = _i32(mb_off)
    L, T, K = ids.shape
    n_mb = mb_off.shape[0] - 1
    hist = np.zeros((n_mb, L, E), dtype=np.int32)
    step = np.zeros((L, E), dtype=np.int64) if want_step else None
    fault = lib().oracle_load_hist(L, T, K, E, n_mb, _p(ids), _p(mb_off), _p(hist), _p(step))
    return hist, step, fault


def quota(c: np.ndarray, slot_expert: np.ndarray, P: int, Ns: int, stop_after: int = 3):
    """O2 for one instance -> quota[S], rank_load[P], slot_off[S+1], (passes, moved), fault."""
    c = _i32(c)
    se = _i32(slot_expert)
    E, S = c.shape[0], P * Ns
    assert se.shape == (S,)
    q = np.zeros(S, dtype=np.int32)
    rl = np.zeros(P, dtype=np.int32)
    so = np.zeros(S + 1, dtype=np.int32)
    stats = np.zeros(2, dtype=np.int32)
    fault = lib().oracle_quota(E, P, Ns, _p(c), _p(se), _p(q), _p(rl), _p(so), stop_after,
                               _p(stats))
    return q, rl, so, (int(stats[0]), int(stats[1])), fault


def check_quota(c, slot_expert, q) -> int:
    c, se, q = _i32(c), _i32(slot_expert), _i32(q)
    return lib().oracle_check_quota(c.shape[0], se.shape[0], _p(c), _p(se), _p(q))


def assign_instance(ids_flat, slot_expert, q, slot_off, E: int, base: int = 0):
    """O3+O4 for one instance -> pair_slot, inv, perm (each [n_pairs]), fault."""
    ids_flat = _i32(ids_flat).ravel()
    se, q, so = _i32(slot_expert), _i32(q), _i32(slot_off)
    n = ids_flat.shape[0]
    ps = np.full(n, -1, dtype=np.int32)
    inv = np.full(n, -1, dtype=np.int32)
    perm = np.full(n, -1, dtype=np.int32)
    fault = lib().oracle_assign_instance(E, se.shape[0], n, base, _p(ids_flat), _p(se), _p(q),
                                         _p(so), _p(ps), _p(inv), _p(perm))
    return ps, inv, perm, fault


def plan(ids, mb_off, hist, slot_expert, P: int, Ns: int, quota_in=None):
    """Whole-step O2+O3+O4 -> dict(quota, rank_load, slot_off, pair_slot, inv, perm, fault)."""
    ids, mb_off, hist, se = _i32(ids), _i32(mb_off), _i32(hist), _i32(slot_expert)
    L, T, K = ids.shape
    n_mb = mb_off.shape[0] - 1
    E = hist.shape[2]
    S = P * Ns
    assert se.shape == (L, S) and hist.shape == (n_mb, L, E)
    qi = None if quota_in is None else _i32(quota_in)
    out = dict(
        quota=np.zeros((n_mb, L, S), dtype=np.int32),
        rank_load=np.zeros((n_mb, L, P), dtype=np.int32),
        slot_off=np.zeros((n_mb, L, S + 1), dtype=np.int32),
        pair_slot=np.full((L, T, K), -1, dtype=np.int32),
        inv=np.full((L, T, K), -1, dtype=np.int32),
        perm=np.full((L, T * K), -1, dtype=np.int32),
    )
    out["fault"] = lib().oracle_plan(L, T, K, E, P, Ns, n_mb, _p(ids), _p(mb_off), _p(hist),
                                     _p(se), _p(qi), _p(out["quota"]), _p(out["rank_load"]),
                                     _p(out["slot_off"]), _p(out["pair_slot"]), _p(out["inv"]),
                                     _p(out["perm"]))
    return out


def gather(perm: np.ndarray, x: np.ndarray, K: int, pair_base: int = 0) -> np.ndarray:
    """O5.  perm: layer-global pair indices of the rows wanted; x: [n_tok, H] rows (any dtype)."""
    perm = _i32(perm).ravel()
    x = np.ascontiguousarray(x)
    row_bytes = x.shape[1] * x.dtype.itemsize
    buf = np.empty((perm.shape[0], x.shape[1]), dtype=x.dtype)
    lib().oracle_gather.argtypes = [C.c_int64, C.c_int, C.c_int64, C.c_int32, C.c_void_p,
                                    C.c_void_p, C.c_void_p]
    lib().oracle_gather(perm.shape[0], K, row_bytes, pair_base, _p(perm), _p(x), _p(buf))
    return buf


def combine(inv: np.ndarray, w: np.ndarray, eo: np.ndarray, act_dtype: int,
            row_base: int = 0) -> np.ndarray:
    """O6.  inv int32 [n_tok,K] layer-global rows, w fp32 [n_tok,K], eo [n_rows,H] (uint16 bf16
    bits when act_dtype == 0, float32 when 1) -> y fp32 [n_tok,H]."""
    inv = _i32(inv)
    w = np.ascontiguousarray(w, dtype=np.float32)
    eo = np.ascontiguousarray(eo)
    assert eo.dtype == (np.uint16 if act_dtype == 0 else np.float32)
    n_tok, K = inv.shape
    H = eo.shape[1]
    y = np.empty((n_tok, H), dtype=np.float32)
    lib().oracle_combine.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int32,
                                     C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib().oracle_combine(n_tok, K, H, act_dtype, row_base, _p(inv), _p(w), _p(eo), _p(y))
    return y


def base_placement(tot: np.ndarray, P: int, Nb: int, Nr: int):
    """O7 for one layer: step totals int64 [E] -> slot_expert int32 [S], fault."""
    tot = np.ascontiguousarray(tot, dtype=np.int64)
    se = np.full(P * (Nb + Nr), -1, dtype=np.int32)
    fault = lib().oracle_base_placement(tot.shape[0], P, Nb, Nr, _p(tot), _p(se))
    return se, fault


def microstep_placement(c: np.ndarray, base_se: np.ndarray, P: int, Nb: int, Nr: int, M: int = 1):
    """O8 for one instance: micro-step loads int32 [E], base placement [S] -> slot_expert [S], fault."""
    c, base_se = _i32(c), _i32(base_se)
    se = np.full(P * (Nb + Nr), -1, dtype=np.int32)
    fault = lib().oracle_microstep_placement(c.shape[0], P, Nb, Nr, M, _p(c), _p(base_se), _p(se))
    return se, fault


def combine_bwd(inv: np.ndarray, w: np.ndarray, dy: np.ndarray, eo: Optional[np.ndarray],
                act_dtype: int, n_rows: int, row_base: int = 0, want_dw: bool = True,
                d_eo_init: Optional[np.ndarray] = None):
    """O9.  inv int32 [n_tok,K] layer-global rows, w fp32 [n_tok,K], dy fp32 [n_tok,H], eo
    [n_rows,H] (uint16 bf16 bits / float32) or None -> d_eo [n_rows,H] (same dtype as eo; rows no
    pair maps to keep d_eo_init or 0), dw fp32 [n_tok,K] (None if not wanted)."""
    inv = _i32(inv)
    w = np.ascontiguousarray(w, dtype=np.float32)
    dy = np.ascontiguousarray(dy, dtype=np.float32)
    n_tok, K = inv.shape
    H = dy.shape[1]
    dt = np.uint16 if act_dtype == 0 else np.float32
    if eo is not None:
        eo = np.ascontiguousarray(eo)
        assert eo.dtype == dt and eo.shape == (n_rows, H)
    d_eo = np.zeros((n_rows, H), dtype=dt) if d_eo_init is None else np.ascontiguousarray(d_eo_init, dtype=dt).copy()
    dw = np.empty((n_tok, K), dtype=np.float32) if (want_dw and eo is not None) else None
    f = lib().oracle_combine_bwd
    f.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int32] + [C.c_void_p] * 6
    f(n_tok, K, H, act_dtype, row_base, _p(inv), _p(w), _p(dy), _p(eo), _p(d_eo), _p(dw))
    return d_eo, dw


def dispatch_bwd(inv: np.ndarray, d_buf: np.ndarray, act_dtype: int, row_base: int = 0) -> np.ndarray:
    """O10.  inv int32 [n_tok,K], d_buf [n_rows,H] (uint16 bf16 bits / float32) -> dx fp32 [n_tok,H]."""
    inv = _i32(inv)
    d_buf = np.ascontiguousarray(d_buf)
    assert d_buf.dtype == (np.uint16 if act_dtype == 0 else np.float32)
    n_tok, K = inv.shape
    H = d_buf.shape[1]
    dx = np.empty((n_tok, H), dtype=np.float32)
    f = lib().oracle_dispatch_bwd
    f.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int32] + [C.c_void_p] * 3
    f(n_tok, K, H, act_dtype, row_base, _p(inv), _p(d_buf), _p(dx))
    return dx


def local_placement(slot_expert: np.ndarray, E: int, P: int, Ns: int, M: int):
    """O11 reduction: real placement [S] -> virtual placement [S*M] (virtual expert e*M+m on virtual
    slot j*M+m when slot j is an allowed host of commodity (e, m)), fault."""
    se = _i32(slot_expert)
    out = np.full(P * Ns * M, -1, dtype=np.int32)
    fault = lib().oracle_local_placement(E, P, Ns, M, _p(se), _p(out))
    return out, fault


def quota_local(w_se: np.ndarray, slot_expert: np.ndarray, P: int, Ns: int, M: int):
    """O11 for one instance: per-source counts int32 [P,E], placement [S] ->
    dict(q_src [M,S], rank_load [P], traffic [M,M], quota_v [S*M], slot_off_v [S*M+1], fault)."""
    w_se, se = _i32(w_se), _i32(slot_expert)
    E, S = w_se.shape[1], P * Ns
    out = dict(q_src=np.zeros((M, S), np.int32), rank_load=np.zeros(P, np.int32),
               traffic=np.zeros((M, M), np.int32), quota_v=np.zeros(S * M, np.int32),
               slot_off_v=np.zeros(S * M + 1, np.int32))
    out["fault"] = lib().oracle_quota_local(E, P, Ns, M, _p(w_se), _p(se), _p(out["q_src"]),
                                            _p(out["rank_load"]), _p(out["traffic"]),
                                            _p(out["quota_v"]), _p(out["slot_off_v"]))
    return out


def replica_search(c_me: np.ndarray, placed_se: np.ndarray, P: int, Nb: int, Nr: int, M: int = 1,
                   a: int = 1, b: int = 0, max_copies: int = 8):
    """O16 for one instance: per-source-machine loads int32 [M,E] (or [E] with M = 1), placement with final
    base slots [S] -> placement with the redundant slots filled by Alg. 2 Stage 3, stats (replicas, F before,
    F after), fault."""
    c_me = _i32(c_me).reshape(M, -1)
    placed_se = _i32(placed_se)
    out = np.full(P * (Nb + Nr), -1, dtype=np.int32)
    stats = np.zeros(3, dtype=np.int64)
    f = lib().oracle_replica_search
    f.argtypes = [C.c_int] * 6 + [C.c_int64, C.c_int64] + [C.c_void_p] * 4
    fault = f(c_me.shape[1], P, Nb, Nr, M, max_copies, a, b, _p(c_me), _p(placed_se), _p(out), _p(stats))
    return out, stats, fault


DEFAULT_LADDER = ((0, 0), (2, 1), (1, 1), (1, 2), (1, 4), (0, 1))   # theta = inf, 2, 1, 1/2, 1/4, 0 as (num, den)


def local_placement_theta(c_v: np.ndarray, slot_expert: np.ndarray, E: int, P: int, Ns: int, M: int,
                          num: int, den: int):
    """O15 member: commodity counts int32 [E*M], real placement [S] -> virtual placement [S*M], fault."""
    c_v, se = _i32(c_v), _i32(slot_expert)
    out = np.full(P * Ns * M, -1, dtype=np.int32)
    f = lib().oracle_local_placement_theta
    f.argtypes = [C.c_int] * 4 + [C.c_int64, C.c_int64] + [C.c_void_p] * 3
    fault = f(E, P, Ns, M, num, den, _p(c_v), _p(se), _p(out))
    return out, fault


def quota_tradeoff(w_se: np.ndarray, slot_expert: np.ndarray, P: int, Ns: int, M: int, a: int, b: int,
                   ladder=DEFAULT_LADDER):
    """O15 for one instance: per-source counts int32 [P,E], placement [S], objective a*L_max + b*C_max ->
    dict(member, F [n_theta], q_src [M,S], rank_load [P], traffic [M,M], quota_v, slot_off_v, se_v, fault)."""
    w_se, se = _i32(w_se), _i32(slot_expert)
    E, S = w_se.shape[1], P * Ns
    num = np.array([t[0] for t in ladder], dtype=np.int64)
    den = np.array([t[1] for t in ladder], dtype=np.int64)
    out = dict(member=np.zeros(1, np.int32), F=np.zeros(len(ladder), np.int64),
               q_src=np.zeros((M, S), np.int32), rank_load=np.zeros(P, np.int32),
               traffic=np.zeros((M, M), np.int32), quota_v=np.zeros(S * M, np.int32),
               slot_off_v=np.zeros(S * M + 1, np.int32), se_v=np.zeros(S * M, np.int32))
    f = lib().oracle_quota_tradeoff
    f.argtypes = [C.c_int] * 4 + [C.c_int64, C.c_int64, C.c_int] + [C.c_void_p] * 12
    out["fault"] = f(E, P, Ns, M, a, b, len(ladder), _p(num), _p(den), _p(w_se), _p(se), _p(out["member"]),
                     _p(out["F"]), _p(out["q_src"]), _p(out["rank_load"]), _p(out["traffic"]),
                     _p(out["quota_v"]), _p(out["slot_off_v"]), _p(out["se_v"]))
    out["member"] = int(out["member"][0])
    return out


def swap_relocation(c_me: np.ndarray, base_se: np.ndarray, P: int, Nb: int, Nr: int, M: int = 1,
                    win: int = 2, max_rounds: int = 16, a: int = 1, b: int = 0):
    """O12 for one instance: per-source-machine loads int32 [M,E] (or [E] with M = 1), base
    placement [S] -> relocated placement [S], stats (rounds, objective before, after), fault."""
    c_me = _i32(c_me).reshape(M, -1)
    base_se = _i32(base_se)
    out = np.full(P * (Nb + Nr), -1, dtype=np.int32)
    stats = np.zeros(3, dtype=np.int64)
    f = lib().oracle_swap_relocation
    f.argtypes = [C.c_int] * 7 + [C.c_int64, C.c_int64] + [C.c_void_p] * 4
    fault = f(c_me.shape[1], P, Nb, Nr, M, win, max_rounds, a, b, _p(c_me), _p(base_se), _p(out), _p(stats))
    return out, stats, fault


def replication(c: np.ndarray, placed_se: np.ndarray, P: int, Nb: int, Nr: int, M: int = 1):
    """O13 for one instance: micro-step loads int32 [E], placement with final base slots [S] ->
    slot_expert [S] with the redundant slots filled by Stage 3, fault."""
    c, placed_se = _i32(c), _i32(placed_se)
    se = np.full(P * (Nb + Nr), -1, dtype=np.int32)
    fault = lib().oracle_replication(c.shape[0], P, Nb, Nr, M, _p(c), _p(placed_se), _p(se))
    return se, fault


def base_placement_machines(tot_me: np.ndarray, P: int, Nb: int, Nr: int, M: int, a: int = 1, b: int = 0):
    """O14 for one layer: step totals per source machine int64 [M,E] -> slot_expert int32 [S], fault."""
    tot_me = np.ascontiguousarray(tot_me, dtype=np.int64).reshape(M, -1)
    se = np.full(P * (Nb + Nr), -1, dtype=np.int32)
    f = lib().oracle_base_placement_machines
    f.argtypes = [C.c_int] * 5 + [C.c_int64, C.c_int64, C.c_void_p, C.c_void_p]
    fault = f(tot_me.shape[1], P, Nb, Nr, M, a, b, _p(tot_me), _p(se))
    return se, fault
