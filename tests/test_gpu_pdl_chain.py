"""FOREMOE_FLAG_PLAN_STABLE behind a chain of overlapping kernels.

The flag lets a data-path kernel fetch its first plan entries (mb_off, inv, w) before its
grid-dependency wait, on the caller's promise that the kernel launched immediately before it does not
write them.  That promise says nothing about the kernel BEFORE that one -- so the library's kernels
release their dependents only after their own wait: in

    [slow kernel that writes w, releasing its dependents early]  ->  foremoe_dispatch  ->
    foremoe_combine(PLAN_STABLE)

the combine must not become resident (and read w) while the writer is still running, although the
dispatch in between, which never touches w, is resident and waiting all that time.  The writer is a
test fixture (tests/pdl_writer.cu): it spins for about a millisecond before it copies the real
weights over a zeroed w.  y is compared with the oracle's combine on the real weights, bit for bit.

What this test is and is not: it pins the documented contract (include/foremoe.h, "Stream order") on the
chain that the contract's wording leaves to the library, eagerly and as a replayed CUDA graph.  It is
not a reproducer: on the B200 / driver 580 box it was written on, the library from before the change
(dependents released ahead of the wait) passed it as well -- a kernel two places down the chain was
never seen running beside the writer there.  The order now holds by construction instead of by that
observation.
"""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest
import torch

from oracle import foremoe_oracle as orc
from paper_2606_11867_b200 import binding as fm
from paper_2606_11867_b200 import runner, synth
from tests import gpu_common as G

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


@pytest.fixture(scope="module")
def writer(tmp_path_factory):
    so = tmp_path_factory.mktemp("pdl") / "libpdl_writer.so"
    subprocess.run([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "-shared", "-Xcompiler", "-fPIC",
                    "-cudart", "static", os.path.join(ROOT, "tests", "pdl_writer.cu"), "-o", str(so)], check=True)
    lib = C.CDLL(str(so))
    lib.slow_copy.argtypes = [C.c_void_p, C.c_void_p, C.c_longlong, C.c_longlong, C.c_void_p]
    return lib


@pytest.mark.parametrize("mode", ["stream", "graph"])
@pytest.mark.parametrize("dispatch_flags", [0, fm.FLAG_PLAN_STABLE])
@pytest.mark.parametrize("sample_len,H", [(48, 2048), (200, 512), (33, 7168)])
def test_combine_plan_stable_behind_writer_and_dispatch(cuda_device, writer, dispatch_flags, sample_len, H, mode):
    """mode "stream": the three launches go to the stream one after the other.  mode "graph": they are
    captured and replayed, where the only edges are the programmatic ones between neighbours (the
    combine has no edge to the writer at all, so the order rests on the dispatch releasing it late)."""
    # micro-steps of one short sample: the dispatch grid is a handful of CTAs, so all three kernels of the
    # chain fit on the machine at once -- the case in which an early-released combine would overlap the writer
    cfg = synth.config(2).scaled(L=2, n_samples=3, sample_len=sample_len, H=H, mb_samples=1)
    ids, w, mb_off, se = G.make_case(cfg)
    ref = G.oracle_plan(ids, mb_off, se, cfg.E, cfg.P, cfg.Ns)
    assert ref["fault"] == 0
    t = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).to(G.DEV)
    w_true = t(w, torch.float32)
    w_d = torch.zeros_like(w_true)
    args = (t(ids, torch.int32), w_d, t(mb_off, torch.int32), t(se, torch.int32))
    sp_d = runner.StepPlan(fm.shape_of(cfg, flags=dispatch_flags), *args)
    sp_d.plan()
    sp_c = runner.StepPlan(fm.shape_of(cfg, flags=fm.FLAG_PLAN_STABLE), *args)      # same w / mb_off, its own flag
    sp_c.inv, sp_c.status = sp_d.inv, sp_d.status
    fm.warmup(sp_d.shape)
    fm.warmup(sp_c.shape)
    s = sp_d.shape
    x = G.activations(cfg, mb_off, range(cfg.n_mb))
    for l in range(cfg.L):
        for i in range(cfg.n_mb):
            a, b = int(mb_off[i]), int(mb_off[i + 1])
            n = b - a
            perm = torch.full((n * s.K,), -5, dtype=torch.int32, device=G.DEV)
            buf = torch.zeros((n * s.K, s.H), dtype=torch.bfloat16, device=G.DEV)
            y = torch.full((n, s.H), float("nan"), dtype=torch.float32, device=G.DEV)

            def chain():        # no sync inside: writer (about 1 ms of spinning, then w), dispatch, combine
                stream = torch.cuda.current_stream().cuda_stream
                assert writer.slow_copy(w_true.data_ptr(), w_d.data_ptr(), w_d.numel(), 2_000_000, stream) == 0
                sp_d.dispatch(l, i, i + 1, x[i], perm, buf)
                sp_c.combine(l, i, i + 1, buf, y)

            if mode == "graph":
                torch.cuda.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g):
                    chain()
            w_d.zero_()
            y.fill_(float("nan"))
            torch.cuda.synchronize()
            if mode == "graph":
                g.replay()
            else:
                chain()
            torch.cuda.synchronize()
            assert torch.equal(w_d, w_true)
            perm_ref = ref["perm"][l, a * s.K:b * s.K]
            assert (perm.cpu().numpy() == perm_ref).all(), ("perm", l, i)
            buf_ref = orc.gather(perm_ref, G.to_bits(x[i]), s.K, pair_base=a * s.K)
            assert (G.to_bits(buf) == buf_ref).all(), ("buf", l, i)
            y_ref = orc.combine(ref["inv"][l, a:b], w[l, a:b], buf_ref, s.act_dtype, row_base=a * s.K)
            bad = int((y.cpu().numpy().view(np.uint32) != y_ref.view(np.uint32)).sum())
            assert bad == 0, f"layer {l} micro-step {i}: {bad} elements of y were combined with stale weights"
    assert sp_d.faults() == 0
