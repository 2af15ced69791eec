"""Sweep the launch parameters of foremoe_dispatch / foremoe_combine on one config (GPU only).

    python -m paper_2606_11867_b200.tune --config 2 --layers 2 [--quick]
    python -m paper_2606_11867_b200.tune --config 2 --layers 1 --samples 32 --bwd      # backward kernels
    python -m paper_2606_11867_b200.tune --config 3 --layers 0 --planner [--machines M] # planner stages, full config

Prints one JSON line per variant: mean CUDA-event time per launch (us), algorithmic GB/s, and
whether the variant's perm / buf / y are bit-identical to the default kernels' outputs.  Also
prints torch fill / copy rates at the instance's size as calibration.  The defaults in
csrc/foremoe_data.cu and csrc/foremoe_combine_async.cu were chosen from this tool's output
(profiles/r01_sweeps.md).
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_11867_b200 import binding as fm
from paper_2606_11867_b200 import synth

KEYS = ["dispatch_impl", "dispatch_u", "dispatch_cta_per_sm", "dispatch_stages", "dispatch_warps",
        "combine_impl", "combine_u", "combine_cta_per_sm", "combine_depth", "combine_threads", "pdl",
        "bwd_depth", "bwd_cta_per_sm"]
DEFAULTS = {"dispatch_impl": -1, "combine_impl": -1, "pdl": 1}


def set_tuning(**kw) -> None:
    """foremoe_debug_set_tuning: sweeps only; unspecified keys return to their defaults."""
    lib = fm.lib()
    lib.foremoe_debug_set_tuning.restype = None
    for i, k in enumerate(KEYS):
        lib.foremoe_debug_set_tuning(i, int(kw.get(k, DEFAULTS.get(k, 0))))


DISPATCH_VARIANTS = [{}] + [{"dispatch_u": u, "dispatch_cta_per_sm": c} for u in (1, 2, 4, 8) for c in (16, 32, 64, 128)] + [
    {"dispatch_cta_per_sm": 4}, {"dispatch_cta_per_sm": 8},
    {"dispatch_impl": 1}, {"dispatch_impl": 1, "dispatch_warps": 4, "dispatch_stages": 3, "dispatch_cta_per_sm": 14},
]
COMBINE_VARIANTS = [{}] + [
    {"combine_impl": 1, "combine_depth": d, "combine_threads": t} for t in (192, 256, 320, 384, 448) for d in (3, 4, 6)]


BWD_VARIANTS = [{}] + [{"bwd_depth": d, "bwd_cta_per_sm": c} for d in (2, 3) for c in (4, 8, 16, 32)]
BWD_NODW_VARIANTS = [{}] + [{"bwd_depth": d, "bwd_cta_per_sm": c} for d in (2, 4) for c in (16, 32)]


def bwd_sweep(wl, cfg, bench) -> None:
    """foremoe_combine_bwd (with and without dw) and foremoe_dispatch_bwd per launch."""
    bpt = bench.bytes_per_token(cfg)
    es = 2 if cfg.act_dtype == synth.ACT_BF16 else 4
    nodw = cfg.H * (4 + es * cfg.K) + 8 * cfg.K
    wl.plan.plan()

    def run(which, kw):
        set_tuning(**kw)
        ev = []
        for r in range(3):
            for (l, i) in wl.instances:
                wl.plan.dispatch(l, i, i + 1, wl.x[i], wl.perm, wl.buf)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                if which == "combine_bwd":
                    wl.plan.combine_bwd(l, i, i + 1, wl.dy, wl.buf, wl.d_buf, wl.dw)
                elif which == "combine_bwd_nodw":
                    wl.plan.combine_bwd(l, i, i + 1, wl.dy, None, wl.d_buf, None)
                else:
                    wl.plan.dispatch_bwd(l, i, i + 1, wl.buf, wl.dx)
                b.record()
                if r > 0:
                    ev.append((a, b, wl.tok[i]))
        torch.cuda.synchronize()
        ms = np.array([a.elapsed_time(b) for a, b, _ in ev])
        n = np.array([t for _, _, t in ev], dtype=np.float64)
        per = nodw if which == "combine_bwd_nodw" else bpt[which]
        print(json.dumps({which: kw or "default", "us": round(float(ms.mean() * 1e3), 1),
                          "gbs": round(float((n * per).sum() / (ms.sum() * 1e-3) / 1e9), 1)}), flush=True)

    for kw in BWD_VARIANTS:
        run("combine_bwd", kw)
    for kw in BWD_NODW_VARIANTS:
        run("combine_bwd_nodw", kw)
    run("dispatch_bwd", {})
    set_tuning()


def planner_times(wl, cfg, M: int) -> None:
    """Whole-step times of the planner stages that run ahead of the data path (all instances of the
    step in one launch each): Stage 1, Alg. 3 Stages 2-3, Alg. 2 Stage 2, and Stage 4 on the result."""
    import dataclasses
    s, dev = wl.shape, wl.dev
    p = wl.plan
    p.load_hist()
    base = torch.empty((s.L, s.S), dtype=torch.int32, device=dev)
    mbp = torch.empty((s.n_mb, s.L, s.S), dtype=torch.int32, device=dev)
    swp = torch.empty_like(mbp)
    rounds = torch.empty((s.n_mb, s.L), dtype=torch.int32, device=dev)
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    s_mb = dataclasses.replace(s, placement_mb_stride=s.L * s.S)
    ws_mb = torch.empty(fm.workspace_bytes(s_mb) + 16, dtype=torch.uint8, device=dev)   # one table set per instance

    def assign_mb(se_mb):
        fm.assign(s_mb, p.ids, p.mb_off, p.hist, se_mb, None, p.quota, p.rank_load, p.slot_off, p.pair_slot,
                  p.inv, ws_mb, st)

    def ratio():
        rl = p.rank_load.float()
        r = (rl.max(-1).values / rl.mean(-1).clamp(min=1e-9))
        return {"median": round(float(r.median()), 4), "mean": round(float(r.mean()), 4), "max": round(float(r.max()), 4)}

    calls = [
        ("foremoe_load_hist", p.load_hist, None),
        ("foremoe_assign (step-level placement from the harness)", p.assign, ratio),
        ("foremoe_base_placement (Stage 1)", lambda: fm.base_placement(s, p.step_hist, base, st), None),
        (f"foremoe_microstep_placement (Alg. 3 Stages 2-3, M={M})", lambda: fm.microstep_placement(s, M, p.hist, base, mbp, st), None),
        ("foremoe_assign on Alg. 3 placements", lambda: assign_mb(mbp), ratio),
        ("foremoe_swap_relocation (Alg. 2 Stage 2, M=1, win=4, <=32 rounds, a=1 b=0)",
         lambda: fm.swap_relocation(s, 1, 4, 32, 1, 0, p.hist, base, swp, rounds, st), None),
        ("foremoe_assign on swap-relocated placements (no replicas)", lambda: assign_mb(swp), ratio),
    ]
    for name, fn, after in calls:
        ts = []
        for r in range(5):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); torch.cuda.synchronize()
            if r >= 2:
                ts.append(a.elapsed_time(b))
        line = {"call": name, "ms": round(float(np.mean(ts)), 3), "instances": cfg.L * cfg.n_mb}
        if after:
            line["lmax_over_lmean"] = after()
        if "swap_relocation" in name:
            line["rounds"] = {"mean": round(float(rounds.float().mean()), 2), "max": int(rounds.max())}
        print(json.dumps(line), flush=True)
    assert int(st.item()) == 0, int(st.item())


def hist_sweep(wl, cfg) -> None:
    """foremoe_load_hist with each k_load_hist mode on the config's trace and on the worst case
    for shared atomics (every pair selects expert 0); results are checked against each other."""
    lib = fm.lib()
    lib.foremoe_debug_set_hist_variant.restype = None
    sp = wl.plan
    names = {0: "plain atomics, 4-byte loads", 1: "warp-aggregated (match.any)",
             2: "plain atomics, 16-byte loads"}
    pairs = cfg.L * cfg.T * cfg.K
    for label, ids in (("config trace", sp.ids), ("all pairs -> expert 0", torch.zeros_like(sp.ids))):
        ref = None
        for mode in (0, 1, 2):
            lib.foremoe_debug_set_hist_variant(mode)
            ts = []
            for r in range(6):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                fm.load_hist(sp.shape, ids, sp.mb_off, sp.hist, sp.step_hist, sp.status)
                b.record(); torch.cuda.synchronize()
                if r >= 2:
                    ts.append(a.elapsed_time(b))
            same = True if ref is None else bool(torch.equal(ref, sp.hist))
            ref = sp.hist.clone() if ref is None else ref
            ms = float(np.mean(ts))
            print(json.dumps({"hist": label, "mode": mode, "what": names[mode], "ms": round(ms, 3),
                              "ids_gbs": round(pairs * 4 / ms / 1e6, 1), "identical": same}), flush=True)
    lib.foremoe_debug_set_hist_variant(2)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--layers", type=int, default=2, help="0 = all layers of the config")
    ap.add_argument("--samples", type=int, default=None, help="fewer samples (config 3: 32)")
    ap.add_argument("--mb-samples", type=int, default=None, help="config 4: samples per micro-step")
    ap.add_argument("--quick", action="store_true")
    ap.add_argument("--hist", action="store_true", help="sweep the k_load_hist modes instead")
    ap.add_argument("--plan", action="store_true", help="time foremoe_load_hist / foremoe_assign only")
    ap.add_argument("--bwd", action="store_true", help="sweep the backward kernels instead")
    ap.add_argument("--planner", action="store_true", help="time the planner stages (placement, relocation, Stage 4)")
    ap.add_argument("--machines", type=int, default=1, help="--planner: machines for Alg. 3")
    args = ap.parse_args()
    import bench
    cfg = synth.config(args.config, mb_samples=args.mb_samples)
    if args.layers > 0 or args.samples:
        cfg = cfg.scaled(L=args.layers if args.layers > 0 else None, n_samples=args.samples)
    dev = torch.device("cuda:0")
    wl = bench.Workload(cfg, dev, "update" if args.bwd else "recompute")
    if args.bwd:
        bwd_sweep(wl, cfg, bench)
        return
    if args.planner:
        print(json.dumps({"workload": bench.workload_name(cfg)}), flush=True)
        planner_times(wl, cfg, args.machines)
        return
    if args.hist:
        hist_sweep(wl, cfg)
        return
    if args.plan:
        for name, fn in (("foremoe_load_hist", wl.plan.load_hist), ("foremoe_assign", wl.plan.assign)):
            ts = []
            for r in range(5):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); fn(); b.record(); torch.cuda.synchronize()
                if r >= 2:
                    ts.append(a.elapsed_time(b))
            print(json.dumps({"call": name, "ms": round(float(np.mean(ts)), 3),
                              "instances": cfg.L * cfg.n_mb, "pairs": cfg.L * cfg.T * cfg.K}), flush=True)
        return
    wl.plan.plan()
    torch.cuda.synchronize()
    bpt = bench.bytes_per_token(cfg)
    tok = max(wl.tok)

    def timeit(which: str, reps: int = 2):
        ev = []
        for r in range(reps + 1):
            for (l, i) in wl.instances:
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                if which == "dispatch":
                    a.record(); wl.plan.dispatch(l, i, i + 1, wl.x[i], wl.perm, wl.buf); b.record()
                else:
                    wl.plan.dispatch(l, i, i + 1, wl.x[i], wl.perm, wl.buf)
                    a.record(); wl.plan.combine(l, i, i + 1, wl.buf, wl.y); b.record()
                if r > 0:
                    ev.append((a, b, wl.tok[i]))
        torch.cuda.synchronize()
        ms = np.array([a.elapsed_time(b) for a, b, _ in ev])
        n = np.array([t for _, _, t in ev], dtype=np.float64)
        return round(float(ms.mean() * 1e3), 1), round(float((n * bpt[which]).sum() / (ms.sum() * 1e-3) / 1e9), 1)

    def loop_time(reps: int = 2):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for r in range(reps + 1):
            if r == 1:
                a.record()
            for (l, i) in wl.instances:
                wl.plan.dispatch(l, i, i + 1, wl.x[i], wl.perm, wl.buf)
                wl.plan.combine(l, i, i + 1, wl.buf, wl.y)
        b.record(); torch.cuda.synchronize()
        ms = a.elapsed_time(b) / reps
        return round(ms * 1e3 / len(wl.instances), 1), round(sum(wl.tok) * cfg.L * (bpt["dispatch"] + bpt["combine"]) / ms / 1e6, 1)

    set_tuning()
    l0, i0 = wl.instances[len(wl.instances) // 2]
    wl.plan.dispatch(l0, i0, i0 + 1, wl.x[i0], wl.perm, wl.buf)
    wl.plan.combine(l0, i0, i0 + 1, wl.buf, wl.y)
    ref = (wl.perm.clone(), wl.buf.clone(), wl.y.clone())

    def same(kw) -> bool:
        set_tuning(**kw)
        wl.perm.fill_(-9); wl.buf.zero_(); wl.y.zero_()
        wl.plan.dispatch(l0, i0, i0 + 1, wl.x[i0], wl.perm, wl.buf)
        wl.plan.combine(l0, i0, i0 + 1, wl.buf, wl.y)
        torch.cuda.synchronize()
        return bool(torch.equal(wl.perm, ref[0]) and torch.equal(wl.buf.view(torch.uint8), ref[1].view(torch.uint8))
                    and torch.equal(wl.y.view(torch.int32), ref[2].view(torch.int32)))

    print(json.dumps({"workload": bench.workload_name(cfg), "tokens_per_instance": tok,
                      "bytes_per_token": bpt}), flush=True)
    # calibration: plain torch fill / copy of the instance's buf size
    nbytes = wl.buf.numel() * wl.buf.element_size()
    other = torch.empty_like(wl.buf)
    for name, fn, moved in (("torch fill_", lambda: wl.buf.view(torch.int32).fill_(1), nbytes),
                            ("torch copy_", lambda: other.copy_(wl.buf), 2 * nbytes)):
        ts = []
        for r in range(8):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); torch.cuda.synchronize()
            if r >= 2:
                ts.append(a.elapsed_time(b))
        print(json.dumps({"calibration": name, "bytes": moved, "us": round(float(np.mean(ts)) * 1e3, 1),
                          "gbs": round(moved / float(np.mean(ts)) / 1e6, 1)}), flush=True)
    del other
    dv = DISPATCH_VARIANTS[:3] if args.quick else DISPATCH_VARIANTS
    cv = COMBINE_VARIANTS[:3] if args.quick else COMBINE_VARIANTS
    for kw in dv:
        ok = same(kw); set_tuning(**kw)
        us, gbs = timeit("dispatch")
        print(json.dumps({"dispatch": kw or "default", "identical": ok, "us": us, "gbs": gbs}), flush=True)
    for kw in cv:
        ok = same(kw); set_tuning(**kw)
        us, gbs = timeit("combine")
        print(json.dumps({"combine": kw or "default", "identical": ok, "us": us, "gbs": gbs}), flush=True)
    for kw in ({}, {"pdl": 0}):
        set_tuning(**kw)
        us, gbs = loop_time()
        print(json.dumps({"loop dispatch+combine": kw or "default", "us_per_instance": us, "gbs": gbs}), flush=True)
    set_tuning()


if __name__ == "__main__":
    main()
