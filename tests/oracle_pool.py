"""CPU-only worker of the whole-step parity test (tests/test_gpu_wholestep.py): runs the oracle
(O1-O6, as it stands, single-threaded C) over whole LAYERS of a step in a pool of processes, one
process per host core, and leaves every integer output plus a 64-bit checksum of every row of
`buf` and `y` in files the parent maps.  Imports numpy and oracle/ only (never torch / CUDA), so a
spawned worker starts in a second.

Row checksum: the row is read as little-endian 64-bit words v_0 .. v_{n-1};
    cs = sum_j v_j * m_j  (mod 2^64),   m_j = (2 j + 1) * 0x9E3779B97F4A7C15  (mod 2^64)
-- position-dependent odd multipliers, so a changed, swapped or shifted word changes the sum.  The
GPU side evaluates the same expression with torch integer ops (int64 wraps the same way)."""
from __future__ import annotations

import os

import numpy as np

GOLD = 0x9E3779B97F4A7C15


def multipliers(n_words: int) -> np.ndarray:
    j = np.arange(n_words, dtype=np.uint64)
    with np.errstate(over="ignore"):
        return (np.uint64(2) * j + np.uint64(1)) * np.uint64(GOLD)


def row_checksums(rows: np.ndarray) -> np.ndarray:
    """rows: [n, row_bytes] any dtype, row_bytes % 8 == 0 -> uint64 [n]."""
    v = np.ascontiguousarray(rows).view(np.uint64).reshape(rows.shape[0], -1)
    m = multipliers(v.shape[1])
    out = np.empty(v.shape[0], dtype=np.uint64)
    with np.errstate(over="ignore"):
        for a in range(0, v.shape[0], 8192):                  # bounded temporaries
            out[a:a + 8192] = (v[a:a + 8192] * m[None, :]).sum(axis=1, dtype=np.uint64)
    return out


def open_arrays(d: str, meta: dict, mode: str = "r+") -> dict:
    L, T, K, S, P, E, n_mb, H = (meta[k] for k in ("L", "T", "K", "S", "P", "E", "n_mb", "H"))
    xdt = np.uint16 if meta["act_dtype"] == 0 else np.float32
    spec = dict(ids=((L, T, K), np.int32), w=((L, T, K), np.float32), x=((T, H), xdt),
                se=((L, S), np.int32), mb_off=((n_mb + 1,), np.int32),
                hist=((n_mb, L, E), np.int32), quota=((n_mb, L, S), np.int32),
                rank_load=((n_mb, L, P), np.int32), slot_off=((n_mb, L, S + 1), np.int32),
                pair_slot=((L, T, K), np.int32), inv=((L, T, K), np.int32), perm=((L, T * K), np.int32),
                cs_buf=((L, T * K), np.uint64), cs_y=((L, T), np.uint64), fault=((L,), np.int32))
    return {k: np.memmap(os.path.join(d, k + ".bin"), dtype=dt, mode=mode, shape=shp)
            for k, (shp, dt) in spec.items()}


def create_arrays(d: str, meta: dict) -> dict:
    return open_arrays(d, meta, mode="w+")


def run_job(args) -> int:
    """Pool entry: (directory, meta, layers); meta["rows"] selects the row work on top of the plan."""
    return run_layers(args, rows=bool(args[1].get("rows", True)))


def run_layers(args, rows: bool = True) -> int:
    """Oracle over the given layers: O1 + O2-O4 per layer; with `rows` also O5 + O6 per instance and a
    checksum per row."""
    d, meta, layers = args
    from oracle import foremoe_oracle as orc
    A = open_arrays(d, meta)
    K, P, Ns, E, n_mb = meta["K"], meta["P"], meta["Ns"], meta["E"], meta["n_mb"]
    mb = np.array(A["mb_off"])
    for l in layers:
        ids_l = np.array(A["ids"][l:l + 1])
        hist, _, f1 = orc.load_hist(ids_l, mb, E, want_step=False)
        plan = orc.plan(ids_l, mb, hist, np.array(A["se"][l:l + 1]), P, Ns)
        A["fault"][l] = f1 | plan["fault"]
        A["hist"][:, l] = hist[:, 0]
        for name in ("quota", "rank_load", "slot_off"):
            A[name][:, l] = plan[name][:, 0]
        for name in ("pair_slot", "inv", "perm"):
            A[name][l] = plan[name][0]
        if not rows:
            continue
        w_l = np.array(A["w"][l])
        for i in range(n_mb):
            a, b = int(mb[i]), int(mb[i + 1])
            if a == b:
                continue
            buf = orc.gather(plan["perm"][0, a * K:b * K], np.array(A["x"][a:b]), K, pair_base=a * K)
            y = orc.combine(plan["inv"][0, a:b], w_l[a:b], buf, meta["act_dtype"], row_base=a * K)
            A["cs_buf"][l, a * K:b * K] = row_checksums(buf)
            A["cs_y"][l, a:b] = row_checksums(y)
    for v in A.values():
        v.flush()
    return len(layers)
