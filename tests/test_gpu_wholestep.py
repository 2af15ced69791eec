"""Whole-step parity of config 2 at full size, in the launch configuration bench.py times
(SURVEY.md sec. 8(d) "Parity coverage at scale"): the oracle runs over the step in a pool of
processes, one per host core (tests/oracle_pool.py; the oracle itself stays single-threaded C), and

  * EVERY integer output of EVERY instance of the step (hist, quota, rank_load, slot_off, pair_slot,
    inv -- 48 layers x 32 micro-steps) is compared element by element;
  * for every instance of every 4th layer (12 x 32 = 384 instances; all 1536 with
    FOREMOE_WHOLESTEP_ALL=1, about 4 minutes of 16-core oracle time) perm is compared element by
    element and a 64-bit checksum of EVERY ROW of buf and of y, computed by both sides, must agree.
"""
import multiprocessing as mp
import os
import shutil
import tempfile

import numpy as np
import pytest
import torch

import bench
from paper_2606_11867_b200 import synth
from tests import oracle_pool as op

pytestmark = pytest.mark.gpu


def _gpu_row_checksums(t: torch.Tensor) -> torch.Tensor:
    """The expression of oracle_pool.row_checksums with torch integer ops (int64 wraps mod 2^64)."""
    v = t.contiguous().view(torch.int64).view(t.shape[0], -1)
    m = torch.from_numpy(op.multipliers(v.shape[1]).view(np.int64)).to(t.device)
    return (v * m[None, :]).sum(dim=1)


def test_config2_whole_step_rows_and_plan(cuda_device):
    cfg = synth.config(2)
    wl = bench.Workload(cfg, cuda_device)
    sp, s = wl.plan, wl.shape
    sp.plan()
    torch.cuda.synchronize()
    assert sp.faults() == 0
    stride = 1 if os.environ.get("FOREMOE_WHOLESTEP_ALL") else 4
    row_layers = list(range(0, s.L, stride))
    meta = dict(L=s.L, T=s.T, K=s.K, S=s.S, P=s.P, E=s.E, n_mb=s.n_mb, H=s.H, Ns=s.Ns, act_dtype=s.act_dtype)
    d = tempfile.mkdtemp(prefix="foremoe_wholestep_")
    try:
        A = op.create_arrays(d, meta)
        A["ids"][:] = sp.ids.cpu().numpy()
        A["w"][:] = sp.w.cpu().numpy()
        A["se"][:] = wl.se_h
        A["mb_off"][:] = wl.mb_off_h
        mb = wl.mb_off_h
        for i in range(s.n_mb):
            a, b = int(mb[i]), int(mb[i + 1])
            A["x"][a:b] = wl.x[i][:b - a].view(torch.int16).cpu().numpy().view(np.uint16)
        A["cs_buf"][:] = 0
        A["cs_y"][:] = 0
        for v in A.values():
            v.flush()
        n_proc = max(1, len(os.sched_getaffinity(0)))
        # every layer gets its plan; the row work (O5 / O6 + checksums) only on row_layers.  Jobs are
        # single layers, row layers first (they are ~30 x longer), handed out dynamically.
        jobs = [(d, dict(meta, rows=True), [l]) for l in row_layers] + \
               [(d, dict(meta, rows=False), [l]) for l in range(s.L) if l not in row_layers]
        with mp.get_context("spawn").Pool(n_proc) as pool:
            done = sum(pool.imap_unordered(op.run_job, jobs))
        assert done == s.L
        A = op.open_arrays(d, meta, mode="r")
        assert (np.array(A["fault"]) == 0).all()
        # every integer output of every instance
        for name in ("hist", "quota", "rank_load", "slot_off", "pair_slot", "inv"):
            got = getattr(sp, name).cpu().numpy()
            bad = np.argwhere(got != np.array(A[name]))
            assert bad.size == 0, (name, len(bad), bad[0])
        # rows: the bench's own buffers and calls, every instance of the row layers
        n_inst = 0
        for l in row_layers:
            perm_ref = torch.from_numpy(np.array(A["perm"][l])).to(cuda_device)
            cs_buf = torch.from_numpy(np.array(A["cs_buf"][l]).view(np.int64)).to(cuda_device)
            cs_y = torch.from_numpy(np.array(A["cs_y"][l]).view(np.int64)).to(cuda_device)
            for i in range(s.n_mb):
                a, b = int(mb[i]), int(mb[i + 1])
                n = b - a
                if n == 0:
                    continue
                wl.buf.view(torch.uint8).fill_(0xAB)
                wl.y.fill_(float("nan"))
                wl.perm.fill_(-5)
                wl.instance(l, i)
                assert torch.equal(wl.perm[:n * s.K], perm_ref[a * s.K:b * s.K]), ("perm", l, i)
                assert torch.equal(_gpu_row_checksums(wl.buf[:n * s.K]), cs_buf[a * s.K:b * s.K]), ("buf rows", l, i)
                assert torch.equal(_gpu_row_checksums(wl.y[:n]), cs_y[a:b]), ("y rows", l, i)
                n_inst += 1
        assert sp.faults() == 0
        print(f"whole step: integer outputs of {s.L * s.n_mb} instances, row checksums of {n_inst} instances "
              f"({n_inst * (s.K + 1) * (int(mb[1]) - int(mb[0]))} rows), {n_proc} oracle processes")
    finally:
        shutil.rmtree(d, ignore_errors=True)

