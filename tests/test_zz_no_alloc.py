"""foremoe_plan_noalloc: the plan for callers that have no device memory to give as workspace.

Why the entry point exists.  foremoe_plan wants a caller-owned scratch buffer, and some callers cannot
produce one where they plan: a component hosted inside an engine whose allocator claimed nearly all of
HBM at start-up (a cudaMalloc from the guest then fails), a plugin whose host permits allocation only
while it initialises, a step loop that will not pay the device-wide sync of cudaMalloc / cudaFree.
foremoe_plan_noalloc keeps the scratch in an 8 MiB array inside the library image instead (one per GPU,
held until the process exits) and refuses shapes that need more.

What is checked here: on two calls in a row -- different traces and different shapes, so the second
call starts on whatever the first left in the shared array -- every output of the new entry point
equals the output of foremoe_plan with a caller-owned workspace, bit for bit (all outputs are integers;
the other GPU tests hold foremoe_plan itself to the oracle).  Plus the refusal of shapes beyond the
limit, which needs no GPU.

The file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide the
other tests) and makes no assumption about what ran before it: it passes alone in a fresh process,
where its first call is also the one that looks up the array's device address, and after the rest of
the suite.
"""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2606_11867_b200 import binding as fm
from paper_2606_11867_b200 import runner, synth

OUTPUTS = ("hist", "step_hist", "quota", "rank_load", "slot_off", "pair_slot", "inv")


def test_shapes_beyond_the_built_in_scratch_are_refused():
    """Config 2 in full needs 26.5 MiB of scratch: the call says so on the host, before it looks at any
    pointer or touches CUDA (all pointers are NULL here), and the binding turns it into a message that
    names both numbers.  A shape that fits gets past the size check (and then trips on the NULLs)."""
    big = fm.Shape(L=48, E=128, K=8, P=8, Nb=16, Nr=2, T=524288, n_mb=32, H=2048)
    assert fm.workspace_bytes(big) > fm.NOALLOC_SCRATCH_BYTES
    assert fm.lib().foremoe_plan_noalloc(C.byref(big.c()), *([None] * 13)) == fm.ERR_WORKSPACE
    with pytest.raises(fm.ForeMoEError, match="built-in array holds 8388608") as ei:
        fm.plan_noalloc(big, *([None] * 11))
    assert ei.value.code == fm.ERR_WORKSPACE
    small = fm.Shape(L=4, E=128, K=8, P=8, Nb=16, Nr=2, T=131072, n_mb=8, H=2048)
    assert fm.workspace_bytes(small) <= fm.NOALLOC_SCRATCH_BYTES
    assert fm.lib().foremoe_plan_noalloc(C.byref(small.c()), *([None] * 13)) == fm.ERR_INVALID_ARG


def _case(cfg, dev):
    """Seeded trace + greedy placement of the config, as device tensors."""
    ids, w, mb_off = synth.gen_trace(cfg)
    ids, w, mb_off = (a.cpu().numpy() for a in (ids, w, mb_off))
    step = np.stack([np.bincount(ids[l].ravel(), minlength=cfg.E) for l in range(cfg.L)]).astype(np.int64)
    se = synth.gen_placement(cfg, step)
    t = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).to(dev)
    return t(ids, torch.int32), t(w, torch.float32), t(mb_off, torch.int32), t(se, torch.int32)


def _both_paths(cfg, dev):
    """The existing path (foremoe_plan, caller-owned workspace) and foremoe_plan_noalloc on the same
    inputs, each into its own poisoned outputs; returns the two result sets and fault words."""
    shape = fm.shape_of(cfg)
    assert fm.workspace_bytes(shape) <= fm.NOALLOC_SCRATCH_BYTES
    ids, w, mb_off, se = _case(cfg, dev)
    ref = runner.StepPlan(shape, ids, w, mb_off, se)
    new = runner.StepPlan(shape, ids, w, mb_off, se)
    for sp, poison in ((ref, -77), (new, -99)):            # unwritten elements would differ
        for n in OUTPUTS:
            getattr(sp, n).fill_(poison)
    ref.plan()
    before = torch.cuda.memory_allocated(dev)
    fm.plan_noalloc(shape, new.ids, new.mb_off, new.slot_expert, None, new.hist, new.step_hist, new.quota,
                    new.rank_load, new.slot_off, new.pair_slot, new.inv, new.status)
    assert torch.cuda.memory_allocated(dev) == before      # the binding takes nothing from torch's pool either
    torch.cuda.synchronize()
    return ref, new


@pytest.mark.gpu
def test_two_calls_in_a_row_equal_the_workspace_path(cuda_device):
    # call 1: config-2-like, 3 layers, ragged micro-steps of 2 800 tokens -> several ranking chunks each
    # call 2: config-5-like (E = 512, K = 10, 32 ranks x 20 slots): other table sizes on the same scratch
    cfgs = [synth.config(2).scaled(L=3, n_samples=12, sample_len=700, H=2048, mb_samples=4),
            synth.config(5).scaled(L=2, n_samples=3, sample_len=3000, H=4096, mb_samples=1)]
    for call, cfg in enumerate(cfgs):
        ref, new = _both_paths(cfg, cuda_device)
        assert ref.faults() == 0 and new.faults() == 0, call
        for n in OUTPUTS:
            a, b = getattr(ref, n), getattr(new, n)
            assert torch.equal(a, b), f"call {call}: {n} differs in {(a != b).sum().item()} elements"
        # the result is a real plan, not two equal poisons: every pair has a row, quotas add up
        assert int(new.inv.min()) >= 0
        assert int(new.quota.sum()) == cfg.L * new.shape.T * cfg.K


@pytest.mark.gpu
def test_same_shape_twice_with_a_new_trace(cuda_device):
    """Back-to-back calls of one shape in one stream with no sync in between: the second call rebuilds
    every table over the first one's, and both results are right."""
    base = synth.config(2).scaled(L=2, n_samples=10, sample_len=333, H=256, mb_samples=3)
    import dataclasses
    cfgs = [base, dataclasses.replace(base, seed=base.seed + 1)]
    shape = fm.shape_of(base)
    plans = []
    for cfg in cfgs:
        ids, w, mb_off, se = _case(cfg, cuda_device)
        ref = runner.StepPlan(shape, ids, w, mb_off, se)
        new = runner.StepPlan(shape, ids, w, mb_off, se)
        ref.plan()
        plans.append((ref, new))
    torch.cuda.synchronize()
    for ref, new in plans:                                  # two noalloc calls enqueued back to back
        fm.plan_noalloc(shape, new.ids, new.mb_off, new.slot_expert, None, new.hist, new.step_hist,
                        new.quota, new.rank_load, new.slot_off, new.pair_slot, new.inv, new.status)
    torch.cuda.synchronize()
    assert not torch.equal(plans[0][0].inv, plans[1][0].inv)         # the two traces do differ
    for call, (ref, new) in enumerate(plans):
        assert new.faults() == 0
        for n in OUTPUTS:
            assert torch.equal(getattr(ref, n), getattr(new, n)), (call, n)
