"""Host logic of the whole-step parity test (no GPU): the process pool of tests/oracle_pool.py gives
the single-process oracle's plan, and the row checksum notices a changed, swapped or shifted word."""
import multiprocessing as mp
import shutil
import tempfile

import numpy as np
import torch

from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import synth
from tests import oracle_pool as op


def test_row_checksum_is_position_sensitive():
    rng = np.random.default_rng(0)
    rows = rng.integers(0, 2 ** 16, size=(5, 64), dtype=np.uint16)
    cs = op.row_checksums(rows)
    # plain definition, word by word, in Python integers
    for r in range(5):
        words = rows[r].view(np.uint64)
        ref = sum(int(v) * (((2 * j + 1) * op.GOLD) % 2 ** 64) for j, v in enumerate(words)) % 2 ** 64
        assert int(cs[r]) == ref
    swapped = rows.copy()
    swapped[0, :4], swapped[0, 4:8] = rows[0, 4:8].copy(), rows[0, :4].copy()      # two 64-bit words exchanged
    assert op.row_checksums(swapped)[0] != cs[0]
    shifted = np.roll(rows, 4, axis=1)
    assert (op.row_checksums(shifted) != cs).all()
    flipped = rows.copy()
    flipped[3, 17] ^= 1
    d = op.row_checksums(flipped) != cs
    assert d.tolist() == [False, False, False, True, False]
    # the torch expression used on the GPU side (int64 wraps the same way)
    v = torch.from_numpy(rows.view(np.int64))
    m = torch.from_numpy(op.multipliers(v.shape[1]).view(np.int64))
    assert ((v * m[None, :]).sum(1).numpy().view(np.uint64) == cs).all()


def test_pool_equals_single_process_oracle():
    cfg = synth.config(2).scaled(L=3, n_samples=8, sample_len=300, H=256, mb_samples=2)
    ids, w, mb_off = synth.gen_trace(cfg, "cpu")
    ids, w, mb_off = ids.numpy(), w.numpy(), mb_off.numpy()
    hist, step, f = orc.load_hist(ids, mb_off, cfg.E)
    se = synth.gen_placement(cfg, step)
    ref = orc.plan(ids, mb_off, hist, se, cfg.P, cfg.Ns)
    x = synth.gen_activations(cfg, cfg.T, 0, "cpu").view(torch.int16).numpy().view(np.uint16)
    meta = dict(L=cfg.L, T=cfg.T, K=cfg.K, S=cfg.S, P=cfg.P, E=cfg.E, n_mb=cfg.n_mb, H=cfg.H, Ns=cfg.Ns,
                act_dtype=cfg.act_dtype)
    d = tempfile.mkdtemp(prefix="foremoe_pool_")
    try:
        A = op.create_arrays(d, meta)
        A["ids"][:], A["w"][:], A["se"][:], A["mb_off"][:], A["x"][:] = ids, w, se, mb_off, x
        A["cs_buf"][:] = 0
        A["cs_y"][:] = 0
        for v in A.values():
            v.flush()
        jobs = [(d, dict(meta, rows=(l != 1)), [l]) for l in range(cfg.L)]
        with mp.get_context("spawn").Pool(2) as pool:
            assert sum(pool.imap_unordered(op.run_job, jobs)) == cfg.L
        A = op.open_arrays(d, meta, mode="r")
        assert (np.array(A["fault"]) == 0).all() and (np.array(A["hist"]) == hist).all()
        for name in ("quota", "rank_load", "slot_off", "pair_slot", "inv", "perm"):
            assert (np.array(A[name]) == ref[name]).all(), name
        K = cfg.K
        for l in (0, 2):
            for i in range(cfg.n_mb):
                a, b = int(mb_off[i]), int(mb_off[i + 1])
                buf = orc.gather(ref["perm"][l, a * K:b * K], x[a:b], K, pair_base=a * K)
                y = orc.combine(ref["inv"][l, a:b], w[l, a:b], buf, cfg.act_dtype, row_base=a * K)
                assert (np.array(A["cs_buf"][l, a * K:b * K]) == op.row_checksums(buf)).all()
                assert (np.array(A["cs_y"][l, a:b]) == op.row_checksums(y)).all()
        assert (np.array(A["cs_buf"][1]) == 0).all()          # plan-only layer: no row work
    finally:
        shutil.rmtree(d, ignore_errors=True)
