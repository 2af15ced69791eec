#!/usr/bin/env python
"""bench.py -- routed tokens/s of the ForeMoE plan + dispatch + combine path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

One "step" = one pass of the whole hot path over one RL step's routing trace: foremoe_load_hist +
foremoe_assign for the whole step, then foremoe_dispatch + foremoe_combine (identity expert:
expert_out = buf) for every (layer, micro-step) instance.  Workload: BASELINE.json configs[1]
(Qwen3-30B-A3B-shaped trace) unless --config says otherwise.  Prints ONE JSON line (rank 0).

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload on this box's host cores: a baseline, not the target.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

from paper_2606_11867_b200 import multi, synth

METRIC = "routed tokens/s (plan+dispatch+combine)"
METRIC_UPDATE = "routed tokens/s (plan + forward dispatch/combine + backward combine_bwd/dispatch_bwd)"
UNIT = "tokens/s"
NOMINAL_HBM_GBS = 8000.0          # BASELINE.json's "~8 TB/s" denominator, context only
FALLBACK_HBM_GBS = 6650.0         # /opt/skills/guides/B200_PROFILING.md fallback


def bytes_per_token(cfg) -> dict:
    """Algorithmic bytes per routed token (DESIGN.md sec. 6 / SURVEY.md sec. 8(d))."""
    es = 2 if cfg.act_dtype == synth.ACT_BF16 else 4
    d = dict(plan=28 * cfg.K, dispatch=es * cfg.H * (1 + cfg.K) + 8 * cfg.K,
             combine=cfg.H * (es * cfg.K + 4) + 8 * cfg.K,
             total=28 * cfg.K + es * cfg.H * (1 + cfg.K) + cfg.H * (es * cfg.K + 4))
    # backward (--stage update): combine_bwd reads dy + K rows of eo, writes K
    # gradient rows (+ inv, w, dw); dispatch_bwd reads K gradient rows, writes dx (+ inv)
    d["combine_bwd"] = cfg.H * (4 + 2 * es * cfg.K) + 12 * cfg.K
    d["dispatch_bwd"] = cfg.H * (es * cfg.K + 4) + 4 * cfg.K
    d["total_update"] = d["total"] + d["combine_bwd"] + d["dispatch_bwd"]
    return d


def workload_name(cfg) -> str:
    dt = "bf16" if cfg.act_dtype == synth.ACT_BF16 else "fp32"
    return (f"config {cfg.cfg_id} ({cfg.name}): L={cfg.L} E={cfg.E} top-{cfg.K} H={cfg.H} {dt}, "
            f"{len(cfg.sample_len)} samples / {cfg.T} tokens in {cfg.n_mb} micro-steps, "
            f"P={cfg.P} ranks x ({cfg.Nb}+{cfg.Nr}) slots")


def measured_peak() -> tuple:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# --------------------------------------------------------------------------------------------
# clocks: sampled DURING the timed region through NVML (what nvidia-smi reads)
# --------------------------------------------------------------------------------------------
class ClockSampler:
    def __init__(self, index: int, period_s: float = 0.1):
        self.index, self.period, self.samples, self.reasons = index, period_s, [], set()
        self.max_mhz, self._stop, self._thr, self.err = None, threading.Event(), None, None

    def _run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {nv.nvmlClocksEventReasonHwSlowdown: "hw_slowdown",
                     nv.nvmlClocksEventReasonHwThermalSlowdown: "hw_thermal_slowdown",
                     nv.nvmlClocksEventReasonSwThermalSlowdown: "sw_thermal_slowdown",
                     nv.nvmlClocksEventReasonSwPowerCap: "sw_power_cap",
                     nv.nvmlClocksEventReasonHwPowerBrakeSlowdown: "hw_power_brake_slowdown",
                     nv.nvmlClocksEventReasonApplicationsClocksSetting: "applications_clocks_setting"}
            while not self._stop.is_set():
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                self._stop.wait(self.period)
        except Exception as e:          # NVML missing: report it, do not fail the bench
            self.err = repr(e)

    def __enter__(self):
        self._thr = threading.Thread(target=self._run, daemon=True)
        self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._thr.join(5)

    def summary(self) -> dict:
        d = {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
             "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
             "samples": len(self.samples)}
        if self.err:
            d["error"] = self.err
        return d


def physical_gpu_index(local_index: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_index])
        except Exception:
            return local_index
    return local_index


# --------------------------------------------------------------------------------------------
# CPU oracle on a bounded sample of the workload (cpu_baseline leg and --impl reference arm)
# --------------------------------------------------------------------------------------------
class OracleSample:
    """`n_mb` micro-steps x `n_layers` layers of the config's recipe, generated on the CPU, run
    through oracle/ (O1..O6) as it stands: single-threaded plain C."""

    def __init__(self, cfg, n_layers: int, n_mb: int):
        from oracle import foremoe_oracle as orc      # test infrastructure: allowed in this leg only
        self.orc = orc
        n_samples = min(len(cfg.sample_len), n_mb * cfg.mb_samples)
        self.cfg = c = cfg.scaled(L=min(n_layers, cfg.L), n_samples=n_samples)
        c.name = cfg.name
        ids, w, mb_off = synth.gen_trace(c, "cpu")
        self.ids, self.w, self.mb_off = ids.numpy(), w.numpy(), mb_off.numpy()
        _, step, _ = orc.load_hist(self.ids, self.mb_off, c.E)
        self.se = synth.gen_placement(c, step)
        self.x = [synth.gen_activations(c, int(self.mb_off[i + 1] - self.mb_off[i]), i, "cpu")
                  for i in range(c.n_mb)]
        self.x = [t.view(torch.int16).numpy().view(np.uint16) if t.dtype == torch.bfloat16
                  else t.numpy() for t in self.x]
        self.routed_tokens = c.T * c.L
        self.desc = (f"{c.L} layer(s) x {c.n_mb} micro-step(s) = {c.L * c.n_mb} instances, "
                     f"{self.routed_tokens} routed tokens of the same recipe, generated on the CPU")

    def step(self) -> float:
        """One pass of the whole path over the sample; returns seconds."""
        orc, c = self.orc, self.cfg
        t0 = time.perf_counter()
        hist, _, f = orc.load_hist(self.ids, self.mb_off, c.E)
        plan = orc.plan(self.ids, self.mb_off, hist, self.se, c.P, c.Ns)
        assert f == 0 and plan["fault"] == 0
        for l in range(c.L):
            for i in range(c.n_mb):
                a, b = int(self.mb_off[i]), int(self.mb_off[i + 1])
                buf = orc.gather(plan["perm"][l, a * c.K:b * c.K], self.x[i], c.K, pair_base=a * c.K)
                orc.combine(plan["inv"][l, a:b], self.w[l, a:b], buf, c.act_dtype, row_base=a * c.K)
        return time.perf_counter() - t0


_POOL_BARRIER = None


def _pool_init(barrier) -> None:
    global _POOL_BARRIER
    _POOL_BARRIER = barrier


def _pool_worker(job):
    """One host core: its own sample of the workload (different samples of the same recipe), generated
    untimed, then one timed pass of the oracle over it, started together with the other workers."""
    cfg_id, mb_samples, seed, n_mb = job
    cfg = synth.config(cfg_id, mb_samples=mb_samples)
    cfg.seed = seed
    samp = OracleSample(cfg, 1, n_mb)
    _POOL_BARRIER.wait()
    t0 = time.time()
    samp.step()
    return samp.routed_tokens, t0, time.time()


def oracle_all_cores(cfg, n_mb_each: int) -> dict:
    """The oracle as it stands (single-threaded C) on every host core at once: one process per core,
    each over its own instances (instances are independent).  Aggregate routed tokens/s
    over the window from the common start to the last finish."""
    import multiprocessing as mp
    n = max(1, len(os.sched_getaffinity(0)))
    ctx = mp.get_context("spawn")              # the parent holds a CUDA context: no fork
    barrier = ctx.Barrier(n)
    jobs = [(cfg.cfg_id, cfg.mb_samples, cfg.seed + 1000 + k, n_mb_each) for k in range(n)]
    with ctx.Pool(n, initializer=_pool_init, initargs=(barrier,)) as pool:
        res = pool.map(_pool_worker, jobs, chunksize=1)
    tokens = sum(r[0] for r in res)
    secs = max(r[2] for r in res) - min(r[1] for r in res)
    return {"value": tokens / secs, "unit": UNIT, "cores": n, "kind": "oracle",
            "sample": f"{n} processes x (1 layer x {n_mb_each} micro-step(s)) = {tokens} routed tokens, "
                      "one single-threaded oracle process per host core, started together",
            "seconds": secs}


def run_reference(args, cfg) -> None:
    """--impl reference: the oracle on host cores, same metric / unit / config."""
    rank, _, world = multi.env_rank()
    if rank != 0:
        return
    n_mb = max(1, min(4, int(60 / max(1, args.steps + args.warmup))))
    samp = OracleSample(cfg, 1, n_mb)
    for _ in range(args.warmup):
        samp.step()
    secs = [samp.step() for _ in range(args.steps)]
    total = float(sum(secs))
    val = samp.routed_tokens * args.steps / total
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16" if cfg.act_dtype == synth.ACT_BF16 else "f32",
        "data": "synthetic", "config": {"workload": workload_name(cfg)},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": "each step = " + samp.desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------
# our arm: everything resident in HBM, C-ABI calls through the binding
# --------------------------------------------------------------------------------------------
class Workload:
    """Device-resident inputs and outputs of one rank's step (inputs are seeded and synthetic:
    recipe in DESIGN.md sec. 4).  Nothing here is timed."""

    def __init__(self, cfg, dev, stage: str = "recompute", machines: int = 0, planner: str = "stage4",
                 objective=None, plan_stable: bool = True, mb_per_call: int = 1):
        from paper_2606_11867_b200 import binding as fm
        from paper_2606_11867_b200 import runner
        self.fm, self.cfg, self.dev = fm, cfg, dev
        # FOREMOE_FLAG_PLAN_STABLE: ids / w / mb_off are uploaded once and inv is written by foremoe_assign
        # only, so no kernel launched right before a data-path call writes the plan arrays
        self.shape = s = fm.shape_of(cfg, flags=fm.FLAG_PLAN_STABLE if plan_stable else 0)
        ids, w, mb_off = synth.gen_trace(cfg, str(dev))
        self.mb_off_h = cfg.mb_off()
        # step-level placement from the step totals (harness-side stand-in for Stages 1-3)
        se0 = torch.full((s.L, s.S), -1, dtype=torch.int32, device=dev)
        self.plan = runner.StepPlan(s, ids, w, mb_off, se0)
        self.plan.load_hist()
        step_hist = self.plan.step_hist.cpu().numpy()
        self.se_h = synth.gen_placement(cfg, step_hist)
        self.plan.slot_expert.copy_(torch.from_numpy(self.se_h))
        self.machines, self.planner = machines, planner
        if planner == "alg2":   # Alg. 1 + Alg. 2 Stages 2-4 on the device (the paper's recompute-stage planner)
            self.plan = None
            M = max(machines, 1)
            self.tok_src_h = synth.gen_tok_src(cfg)
            a, b = objective if objective else (1, 0)
            self.plan = runner.Alg2StepPlan(s, M, a, b, ids, w, mb_off, torch.from_numpy(self.tok_src_h).to(dev))
            self.real_shape, self.shape = s, self.plan.shape
        elif planner == "full":   # Stages 1-4 on the device: the harness placement above is not used
            self.plan = None
            self.plan = runner.PlannerStepPlan(s, max(machines, 1), ids, w, mb_off)
            self.shape = self.plan.shape
        elif machines:        # per-source, multi-machine Stage 4: commodity plan
            self.tok_src_h = synth.gen_tok_src(cfg)
            se_dev = self.plan.slot_expert
            self.plan = None
            src = torch.from_numpy(self.tok_src_h).to(dev)
            if objective:     # Eq.(10): F = a L_max + b C_max over the threshold ladder (reading 39)
                self.plan = runner.TradeoffStepPlan(s, machines, objective[0], objective[1], ids, w, mb_off, se_dev, src)
            else:             # hard locality (reading 30)
                self.plan = runner.LocalStepPlan(s, machines, ids, w, mb_off, se_dev, src)
            self.real_shape, self.shape = s, self.plan.shape      # same K, H, T, n_mb; E, Nb, Nr x M
        # one data-path call covers `mb_per_call` consecutive micro-steps of a layer (ranged calls of the
        # C ABI; 1 = the order a training loop issues them, the headline).  Call g = micro-steps calls[g].
        tok_mb = [int(self.mb_off_h[i + 1] - self.mb_off_h[i]) for i in range(s.n_mb)]
        self.calls = [(i0, min(i0 + mb_per_call, s.n_mb)) for i0 in range(0, s.n_mb, mb_per_call)]
        tok = [sum(tok_mb[i0:i1]) for (i0, i1) in self.calls]
        self.tok = tok
        if mb_per_call == 1:
            self.x = [synth.gen_activations(cfg, max(n, 1), i, str(dev)) for i, n in enumerate(tok)]
        else:
            self.x = [torch.cat([synth.gen_activations(cfg, max(tok_mb[i], 1), i, str(dev))[:tok_mb[i]]
                                 for i in range(i0, i1)] + [torch.zeros((1, s.H), dtype=s.act_torch_dtype, device=dev)])
                      for (i0, i1) in self.calls]
        mx = max(max(tok), 1)
        self.buf = torch.empty((mx * s.K, s.H), dtype=s.act_torch_dtype, device=dev)
        self.y = torch.empty((mx, s.H), dtype=torch.float32, device=dev)
        self.perm = torch.empty((mx * s.K,), dtype=torch.int32, device=dev)
        self.instances = [(l, g) for l in range(s.L) for g in range(len(self.calls)) if tok[g] > 0]
        self.routed_tokens = sum(tok) * s.L
        self.stage = stage
        n_lad = len(runner.DEFAULT_LADDER) if (objective and machines and planner not in ("full", "alg2")) else 0
        if planner == "alg2":
            n_lad = len(self.plan.ladder)
        # foremoe_plan (given placement: default and LocalStepPlan) launches 7 kernels; the planners that derive
        # the placement from the histogram call foremoe_load_hist (2) + foremoe_assign (6)
        fused = planner == "stage4" and not n_lad
        self.launches_per_step = ((7 if fused else 8) + (3 if machines and planner != "full" else 0) + (2 if planner == "full" else 0)
                                  + n_lad * 5 + (1 if n_lad else 0) + (4 if planner == "alg2" else 0)
                                  + (4 if stage == "update" else 2) * len(self.instances))
        if stage == "update":          # forward + backward of every instance
            self.dy = torch.randn((mx, s.H), dtype=torch.float32, device=dev,
                                  generator=torch.Generator(device=dev).manual_seed(cfg.seed + 11))
            self.d_buf = torch.empty_like(self.buf)
            self.dx = torch.empty_like(self.y)
            self.dw = torch.empty((s.L, s.T, s.K), dtype=torch.float32, device=dev)

    def instance(self, l: int, g: int, ev=None):
        """The data path of one instance (call g of layer l); ev (optional) collects CUDA events between the calls."""
        p = self.plan.data_path()          # binding.DataPath: the plan's arguments marshalled once
        i0, i1 = self.calls[g]
        if ev is None:
            p.dispatch(l, i0, i1, self.x[g], self.perm, self.buf)
            p.combine(l, i0, i1, self.buf, self.y)
            if self.stage == "update":
                p.combine_bwd(l, i0, i1, self.dy, self.buf, self.d_buf, self.dw)
                p.dispatch_bwd(l, i0, i1, self.d_buf, self.dx)
            return

        def mark():
            ev.append(torch.cuda.Event(enable_timing=True))
            ev[-1].record()

        mark()
        p.dispatch(l, i0, i1, self.x[g], self.perm, self.buf)
        mark()
        p.combine(l, i0, i1, self.buf, self.y)
        mark()
        if self.stage == "update":
            p.combine_bwd(l, i0, i1, self.dy, self.buf, self.d_buf, self.dw)
            mark()
            p.dispatch_bwd(l, i0, i1, self.d_buf, self.dx)
            mark()

    def step(self, probes=None, stride: int = 0):
        """One pass of the whole path.  Layers outer, micro-steps inner: consecutive launches read
        different x buffers, so no call finds its input left in L2 by the previous one."""
        p = self.plan
        if probes is not None:
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            e0.record()
        p.plan()
        if probes is not None:
            e1.record()
            probes["plan"].append((e0, e1, self.cfg.T * self.cfg.L))
        run = None                       # an open run of un-probed instances: (start event, tokens so far)
        for n, (l, i) in enumerate(self.instances):
            if probes is not None and stride and n % stride == 0:
                a = []
                self.instance(l, i, a)
                for j, name in enumerate(("dispatch", "combine", "combine_bwd", "dispatch_bwd")[:len(a) - 1]):
                    probes[name].append((a[j], a[j + 1], self.tok[i]))
                if stride >= 4:          # the stride - 1 instances up to the next probe run back to back, un-probed:
                    run = [a[-1], 0]     # one pair of events around the whole run gives the data path's rate IN the loop
            else:
                self.instance(l, i)
                if run is not None:
                    run[1] += self.tok[i]
                    if n % stride == stride - 1:
                        e = torch.cuda.Event(enable_timing=True)
                        e.record()
                        probes["run"].append((run[0], e, run[1]))
                        run = None

    def capture_graph(self):
        """Capture the per-instance loop (dispatch + combine of every instance) into ONE CUDA graph:
        for small micro-steps the loop is launch-bound on the host otherwise."""
        self.step()                                   # all lazy one-time set-up happens before capture
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            for (l, i) in self.instances:
                self.instance(l, i)
        self.graph = g

    def step_graph(self):
        self.plan.plan()
        self.graph.replay()

    def setup_streams(self, n: int):
        """Independent instances on `n` streams (each with its own perm / buf / y / gradient buffers):
        the library is re-entrant per stream and (micro-step, layer) instances are independent
        (PAPER.md:144, :417), so the ramp and drain of one launch overlap another stream's kernel."""
        self.streams = [torch.cuda.Stream() for _ in range(n)]
        names = ["perm", "buf", "y"] + (["d_buf", "dx"] if self.stage == "update" else [])
        self.stream_bufs = [{k: (getattr(self, k) if j == 0 else torch.empty_like(getattr(self, k))) for k in names}
                            for j in range(n)]

    def step_streams(self):
        main = torch.cuda.current_stream()
        self.plan.plan()
        ready = torch.cuda.Event()
        ready.record(main)
        for j, st in enumerate(self.streams):
            st.wait_event(ready)
            with torch.cuda.stream(st):
                for k, v in self.stream_bufs[j].items():
                    setattr(self, k, v)
                for (l, i) in self.instances[j::len(self.streams)]:
                    self.instance(l, i)
        for k, v in self.stream_bufs[0].items():
            setattr(self, k, v)
        for st in self.streams:
            done = torch.cuda.Event()
            done.record(st)
            main.wait_event(done)

    def release(self):
        self.plan = self.x = self.buf = self.y = self.perm = None
        self.dy = self.d_buf = self.dx = self.dw = None
        torch.cuda.empty_cache()


def capture_instance(wl: "Workload", inst) -> tuple:
    """After the timed region: run one instance of the timed configuration once more (same buffers,
    same calls) and bring its inputs and outputs to the host for verify_against_oracle."""
    l, i = inst
    s = wl.shape
    a, b = int(wl.mb_off_h[i]), int(wl.mb_off_h[i + 1])
    n = b - a
    wl.instance(l, i)
    torch.cuda.synchronize()
    bits = lambda t: (t.view(torch.int16).cpu().numpy().view(np.uint16) if t.dtype == torch.bfloat16
                      else t.cpu().numpy())
    return (dict(l=l, i=i, a=a, K=s.K, act_dtype=s.act_dtype), wl.plan.inv[l, a:b].cpu().numpy(),
            wl.plan.w[l, a:b].cpu().numpy(), bits(wl.x[i][:n]), wl.perm[:n * s.K].cpu().numpy(),
            bits(wl.buf[:n * s.K]), wl.y[:n].cpu().numpy())


def verify_against_oracle(meta, inv, w, x, perm, buf, y) -> dict:
    """cpu_baseline leg only: the captured instance's perm / buf / y against O5 / O6, bit for bit (the
    plan itself, inv, is compared with the oracle by the tests; here it is checked to be a bijection
    consistent with perm)."""
    from oracle import foremoe_oracle as orc      # test infrastructure: allowed in this leg only
    K, base = meta["K"], meta["a"] * meta["K"]
    ok_perm = bool((perm[inv.reshape(-1) - base] == np.arange(base, base + inv.size)).all())
    buf_ref = orc.gather(perm, x, K, pair_base=base)
    ok_buf = bool((buf_ref == buf).all())
    y_ref = orc.combine(inv, w, buf_ref, meta["act_dtype"], row_base=base)
    ok_y = bool((y_ref.view(np.uint32) == y.view(np.uint32)).all())
    assert ok_perm and ok_buf and ok_y, ("timed configuration disagrees with the oracle", ok_perm, ok_buf, ok_y)
    return {"instance": [meta["l"], meta["i"]], "perm": ok_perm, "buf_bit_exact": ok_buf, "y_bit_exact": ok_y,
            "against": "oracle O5/O6 after the timed region"}


def probe_stats(probes, bpt) -> dict:
    out = {}
    for name, lst in probes.items():
        if not lst:
            continue
        ms = np.array([a.elapsed_time(b) for a, b, _ in lst])
        toks = np.array([n for _, _, n in lst], dtype=np.float64)
        gbs = float((toks * bpt[name]).sum() / (ms.sum() * 1e-3) / 1e9)
        out[name] = {"launches_timed": len(lst), "avg_ms": float(ms.mean()), "gbs": gbs,
                     "bytes_per_token": bpt[name]}
    return out


def run_e2e(args, cfg, wl: "Workload", dev) -> dict:
    """The same step through foremoe_step_host: HOST (pinned) buffers in, plan + y out, every
    host<->device copy inside the timed region."""
    fm, s = wl.fm, wl.shape
    pin = lambda t: t.contiguous().cpu().pin_memory()
    ids_h, w_h = pin(wl.plan.ids), pin(wl.plan.w)
    mb_h = torch.from_numpy(wl.mb_off_h.copy())
    se_h = torch.from_numpy(wl.se_h.copy())
    x_h = torch.empty((s.T, s.H), dtype=s.act_torch_dtype).pin_memory()
    for i, n in enumerate(wl.tok):
        if n:
            x_h[int(wl.mb_off_h[i]):int(wl.mb_off_h[i + 1])].copy_(wl.x[i][:n])
    routed = wl.routed_tokens
    n_inst = len(wl.instances)
    wl.release()
    q_h = torch.empty((s.n_mb, s.L, s.S), dtype=torch.int32).pin_memory()
    rl_h = torch.empty((s.n_mb, s.L, s.P), dtype=torch.int32).pin_memory()
    so_h = torch.empty((s.n_mb, s.L, s.S + 1), dtype=torch.int32).pin_memory()
    y_h = torch.empty((s.T, s.H), dtype=torch.float32).pin_memory()
    st_h = torch.zeros(1, dtype=torch.int32).pin_memory()
    arena = torch.empty(fm.step_host_arena_bytes(s, mb_h) + 256, dtype=torch.uint8, device=dev)
    arena = arena[(-arena.data_ptr()) % 256:]
    h2d = ids_h.numel() * 4 + w_h.numel() * 4 + mb_h.numel() * 4 + se_h.numel() * 4 \
        + x_h.numel() * x_h.element_size()
    d2h = (q_h.numel() + rl_h.numel() + so_h.numel() + 1) * 4 + s.L * y_h.numel() * 4
    call = lambda: fm.step_host(s, ids_h, w_h, mb_h, se_h, x_h, q_h, rl_h, so_h, y_h, arena, st_h)
    steps = max(1, min(args.steps, args.e2e_steps))
    call()                                            # warm-up (also first-touch of the arena)
    multi.barrier(dev); torch.cuda.synchronize()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        call()                                        # synchronises before returning
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    assert int(st_h[0]) == 0, f"device fault bits {int(st_h[0])}"
    ms_max, units = multi.aggregate(ms, routed * steps, dev)
    return {"value": units / (ms_max * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
            "d2h_bytes_per_step": int(d2h), "steps": steps, "ms_per_step": ms_max / steps,
            "api": "foremoe_step_host (pinned host buffers; x up once per micro-step, y of every "
                   "instance down)", "gpu_launches": steps * (6 + 2 * n_inst)}


def run_ours(args, cfg) -> None:
    rank, local_rank, world = multi.env_rank()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback exists)"
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    multi.init("nccl", dev)
    cfg.seed = multi.shard_seed(cfg.seed, rank)          # each rank: its own step (weak scaling)
    objective = tuple(int(v) for v in args.objective.split(",")) if args.objective else None
    wl = Workload(cfg, dev, args.stage, args.machines, args.planner, objective, not args.strict_order,
                  args.mb_per_call)
    bpt = bytes_per_token(cfg)
    upd = args.stage == "update"
    total_bpt = bpt["total_update"] if upd else bpt["total"]
    peak, peak_src = measured_peak()

    if args.graph:
        wl.capture_graph()
    if args.streams > 1:
        wl.setup_streams(args.streams)
    for _ in range(args.warmup):
        wl.step_streams() if args.streams > 1 else wl.step()
    torch.cuda.synchronize()
    assert wl.plan.faults() == 0
    probes = {"plan": [], "dispatch": [], "combine": [], "combine_bwd": [], "dispatch_bwd": [], "run": []}
    if args.graph or args.streams > 1:
        # per-kernel probes cannot sit inside a graph / between concurrent streams: one extra, untimed step
        wl.step(probes, args.probe_stride)
        torch.cuda.synchronize()
    multi.barrier(dev); torch.cuda.synchronize()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    with ClockSampler(physical_gpu_index(local_rank)) as clk:
        e0.record()
        for _ in range(args.steps):
            if args.graph:
                wl.step_graph()
            elif args.streams > 1:
                wl.step_streams()
            else:
                wl.step(probes, args.probe_stride)
        e1.record()
        torch.cuda.synchronize()
    multi.barrier(dev)
    ms = e0.elapsed_time(e1)
    assert wl.plan.faults() == 0
    ms_max, units = multi.aggregate(ms, wl.routed_tokens * args.steps, dev)
    value = units / (ms_max * 1e-3)
    launches = wl.launches_per_step * args.steps
    bpt["run"] = total_bpt - bpt["plan"]          # a run = whole instances: every data-path kernel of the stage
    kern = probe_stats(probes, bpt)
    in_loop = kern.pop("run", None)
    dom = "combine" if bpt["combine"] >= bpt["dispatch"] else "dispatch"
    if upd:
        dom = "combine_bwd"
    traffic, traffic_src = None, None
    tp = os.path.join(ROOT, "profiles", "traffic.json")      # written from the committed ncu capture
    if os.path.exists(tp):
        try:
            tj = json.load(open(tp))
            traffic = tj.get(f"config{cfg.cfg_id}", {}).get(dom)
            if traffic is not None:
                traffic_src = "stored constant, NOT measured in this run: " + tj.get("_source", "profiles/traffic.json")
        except Exception:
            traffic = None
    probed = kern.get(dom, {"gbs": None, "avg_ms": None})      # absent with --probe-stride 0 (diagnostic lines)
    roofline = {"bound": "hbm", "kernel": f"foremoe_{dom}",
                "achieved": probed["gbs"], "peak": peak, "unit": "GB/s",
                "frac": probed["gbs"] / peak if probed["gbs"] else None, "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": peak_src,
                "bytes_per_launch": bpt[dom] * max(wl.tok), "avg_launch_ms": probed["avg_ms"],
                "whole_path_gbs": value / world * total_bpt / 1e9,
                "whole_path_frac": value / world * total_bpt / 1e9 / peak,
                "whole_path_frac_of_nominal_8TBs": value / world * total_bpt / 1e9 / NOMINAL_HBM_GBS,
                "kernels": kern}
    if in_loop:
        # the same kernels between launches of their own kind, no event inside: runs of (probe stride - 1) whole
        # instances, one pair of CUDA events around each run, inside the timed region
        roofline["data_path_in_loop"] = {"gbs": in_loop["gbs"], "frac": in_loop["gbs"] / peak,
                                         "runs_timed": in_loop["launches_timed"], "avg_run_ms": in_loop["avg_ms"],
                                         "bytes_per_token": in_loop["bytes_per_token"]}
    clocks = clk.summary()
    # load balance of the plan (not timed): per instance max rank load / mean rank load, against the
    # natural placement (expert e on rank e // Nb, no replicas) -- PAPER.md:503-507 reports this ratio
    rl = wl.plan.rank_load.float()
    live = rl.sum(-1) > 0
    ratio = (rl.max(-1).values / rl.mean(-1).clamp(min=1e-9))[live]
    virt = args.planner == "alg2" or (args.machines and args.planner != "full")
    Mv = max(args.machines, 1)
    hist_real = wl.plan.hist.view(cfg.n_mb, cfg.L, cfg.E, Mv).sum(-1) if virt else wl.plan.hist
    nat = hist_real.float().view(cfg.n_mb, cfg.L, cfg.P, cfg.Nb).sum(-1)
    nratio = (nat.max(-1).values / nat.mean(-1).clamp(min=1e-9))[live]
    balance = {"lmax_over_lmean": {"max": float(ratio.max()), "mean": float(ratio.mean()),
                                   "median": float(ratio.median())},
               "natural_placement": {"max": float(nratio.max()), "mean": float(nratio.mean()),
                                     "median": float(nratio.median())}}

    if virt:
        tr = wl.plan.traffic.double()
        tot = tr.sum((-1, -2)).clamp(min=1)
        cross = (tot - tr.diagonal(dim1=-2, dim2=-1).sum(-1)) / tot
        off = tr.clone()
        off.diagonal(dim1=-2, dim2=-1).zero_()
        balance["machines"] = Mv
        if args.planner == "alg2":
            balance["alg2"] = {"swaps_mean": float(wl.plan.swaps[live].float().mean()),
                               "replicas_mean": float(wl.plan.replicas[live].float().mean())}
        if objective or args.planner == "alg2":
            balance["objective"] = {"a": wl.plan.a, "b": wl.plan.b,
                                    "members_chosen": torch.bincount(wl.plan.member[live].flatten().long(),
                                                                     minlength=len(wl.plan.ladder)).tolist(),
                                    "ladder": [list(t) for t in wl.plan.ladder]}
        balance["cross_machine_fraction"] = {"mean": float(cross[live].mean()), "max": float(cross[live].max())}
        balance["c_max_tokens"] = {"median": float(off.amax((-1, -2))[live].median()), "max": float(off.max())}
    line = {
        "metric": METRIC_UPDATE if upd else METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16" if cfg.act_dtype == synth.ACT_BF16 else "f32", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "parallelism": f"{world} independent shard(s), no collective",
                   "l2": "inputs larger than L2: every instance moves >= 1 GB and consecutive "
                         "launches read different x buffers; no flush needed",
                   "plan_stable_flag": not args.strict_order,
                   **({"mb_per_call": args.mb_per_call} if args.mb_per_call != 1 else {}),
                   "stage": args.stage, "machines": args.machines, "planner": args.planner,
                   **({"objective": args.objective} if args.objective else {}), "bytes_per_routed_token": total_bpt,
                   **({"sweep_tuning": args.tune} if args.tune else {}),
                   "launch": ("cuda graph replay of the instance loop" if args.graph else
                              f"{args.streams} streams, independent instances interleaved" if args.streams > 1
                              else "stream launches")},
        "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "balance": balance,
    }
    verify = None
    if (rank == 0 and world == 1 and not args.no_cpu_baseline and not upd and not args.machines
            and args.planner == "stage4" and args.mb_per_call == 1):
        verify = capture_instance(wl, wl.instances[len(wl.instances) // 2])
    if not args.no_e2e and not upd and not args.machines and args.planner == "stage4" and args.mb_per_call == 1:
        line["e2e"] = run_e2e(args, cfg, wl, dev)
    else:
        wl.release()
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not upd:
        n_samp = args.cpu_sample_mb
        if n_samp <= 0:     # ~30 GB of algorithmic bytes = ~15 s for the single-threaded oracle
            per_mb = bpt["total"] * max(1, cfg.T // cfg.n_mb)
            n_samp = int(max(1, min(cfg.n_mb, round(30e9 / per_mb))))
        samp = OracleSample(cfg, 1, n_samp)
        secs = samp.step()
        line["cpu_baseline"] = {"value": samp.routed_tokens / secs, "unit": UNIT, "cores": 1,
                                "kind": "oracle", "sample": samp.desc, "seconds": secs}
        del samp
        if not args.no_cpu_all_cores:
            line["cpu_baseline"]["all_cores"] = oracle_all_cores(cfg, max(1, n_samp // 4))
        if verify is not None:
            line["verified"] = verify_against_oracle(*verify)
    headline = (args.config == 2 and args.mb_samples is None and not args.layers and not upd and not args.machines
                and args.planner == "stage4" and args.mb_per_call == 1 and not args.graph and args.streams == 1
                and not args.tune and not args.strict_order)
    if rank == 0 and world == 1 and headline and not args.no_other_configs:
        del wl
        torch.cuda.empty_cache()
        line["other_configs"] = run_other_configs(args, dev, physical_gpu_index(local_rank), peak)
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        torch.distributed.destroy_process_group()


OTHER_CONFIGS = [(1, None), (3, None), (5, None), (4, 1), (4, 8), (4, 64)]     # (BASELINE.json config, samples per micro-step)


def run_other_config(cfg, dev, gpu_index: int, peak: float, steps: int, warmup: int, probe_stride: int) -> dict:
    """One of the non-headline configs of BASELINE.json, timed like the headline (warm-up, CUDA events around
    `steps` whole steps of foremoe_plan + dispatch + combine of every instance, clocks sampled during the
    timed region, one instance of the timed configuration checked against the oracle afterwards), reported
    as a compact record.  Runs after the headline's timed region and legs, on released memory."""
    wl = Workload(cfg, dev)
    bpt = bytes_per_token(cfg)
    for _ in range(warmup):
        wl.step()
    torch.cuda.synchronize()
    assert wl.plan.faults() == 0
    probes = {"plan": [], "dispatch": [], "combine": [], "combine_bwd": [], "dispatch_bwd": [], "run": []}
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    with ClockSampler(gpu_index) as clk:
        e0.record()
        for _ in range(steps):
            wl.step(probes, probe_stride)
        e1.record()
        torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    assert wl.plan.faults() == 0
    value = wl.routed_tokens * steps / (ms * 1e-3)
    bpt["run"] = bpt["total"] - bpt["plan"]
    kern = probe_stats(probes, bpt)
    kern.pop("run", None)
    rl = wl.plan.rank_load.float()
    live = rl.sum(-1) > 0
    ratio = (rl.max(-1).values / rl.mean(-1).clamp(min=1e-9))[live]
    nat = wl.plan.hist.float().view(cfg.n_mb, cfg.L, cfg.P, cfg.Nb).sum(-1)
    nratio = (nat.max(-1).values / nat.mean(-1).clamp(min=1e-9))[live]
    out = {"workload": workload_name(cfg), "value": value, "unit": UNIT, "steps": steps, "warmup": warmup,
           "ms_per_step": ms / steps, "dtype": "bf16" if cfg.act_dtype == synth.ACT_BF16 else "f32",
           "bytes_per_routed_token": bpt["total"], "whole_path_gbs": value * bpt["total"] / 1e9,
           "whole_path_frac": value * bpt["total"] / 1e9 / peak,
           "gpu_launches": wl.launches_per_step * steps,
           "kernels": {k: {"avg_ms": v["avg_ms"], "gbs": v["gbs"], "frac": v["gbs"] / peak,
                           "launches_timed": v["launches_timed"]} for k, v in kern.items()},
           "balance": {"lmax_over_lmean": {"max": float(ratio.max()), "mean": float(ratio.mean()),
                                           "median": float(ratio.median())},
                       "natural_placement": {"max": float(nratio.max()), "mean": float(nratio.mean()),
                                             "median": float(nratio.median())}},
           "clocks": clk.summary()}
    verify = capture_instance(wl, wl.instances[len(wl.instances) // 2])
    wl.release()
    out["verified"] = verify_against_oracle(*verify)
    return out


def run_other_configs(args, dev, gpu_index: int, peak: float) -> dict:
    """north_star names five configs and a micro-step size sweep "at each size": the default run reports them
    all.  A failure in one of them is recorded in its entry and never costs the headline line."""
    out = {}
    for cfg_id, mb in OTHER_CONFIGS:
        key = str(cfg_id) if mb is None else f"{cfg_id}@{mb}"
        try:
            cfg = synth.config(cfg_id, mb_samples=mb)
            out[key] = run_other_config(cfg, dev, gpu_index, peak, max(2, min(args.steps, 3)), 3, args.probe_stride)
        except Exception as e:      # noqa: BLE001 -- report, do not lose the headline
            out[key] = {"error": f"{type(e).__name__}: {e}"[:300]}
        torch.cuda.empty_cache()
    return out


TUNING_KEYS = ["dispatch_impl", "dispatch_u", "dispatch_cta_per_sm", "dispatch_stages", "dispatch_warps",
               "combine_impl", "combine_u", "combine_cta_per_sm", "combine_depth", "combine_threads", "pdl",
               "bwd_depth", "bwd_cta_per_sm", "bwd_impl", "hist_variant"]      # DataTuning, declaration order


def apply_tuning(spec: str) -> None:
    """Sweep runs: switch the binding to libforemoe_tuning.so and set the named launch parameters."""
    from paper_2606_11867_b200 import binding as fm
    fm.LIB_PATH = os.path.join(fm.HERE, "libforemoe_tuning.so")
    lib = fm.lib()
    lib.foremoe_tuning_set.restype = None
    for kv in spec.split(","):
        k, v = kv.split("=")
        lib.foremoe_tuning_set(TUNING_KEYS.index(k.strip()), int(v))


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-5)")
    ap.add_argument("--mb-samples", type=int, default=None, help="config 4: samples per micro-step")
    ap.add_argument("--layers", type=int, default=None, help="debug: fewer layers (INVALID as a bench value)")
    ap.add_argument("--probe-stride", type=int, default=32,
                    help="CUDA-event brackets around every n-th instance's dispatch / combine launch")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-sample-mb", type=int, default=0,
                    help="micro-steps (x 1 layer) of the workload the oracle is timed on; 0 = as many as make "
                         "about 15 s of CPU work (the oracle moves ~2 GB/s of algorithmic bytes on one core)")
    ap.add_argument("--graph", action="store_true",
                    help="replay the per-instance loop as one CUDA graph (per-kernel probes are then "
                         "taken in an extra untimed step)")
    ap.add_argument("--stage", default="recompute", choices=["recompute", "update"],
                    help="recompute = the headline forward path; update = forward + backward of every "
                         "instance (policy-update stage, PAPER.md:241; no e2e / oracle legs)")
    ap.add_argument("--machines", type=int, default=0,
                    help="M > 0: per-source, locality-aware Stage 4 over M machines of P/M ranks "
                         "(commodity plan, SURVEY.md sec. 8(f).1); the data path is unchanged")
    ap.add_argument("--objective", default="",
                    help="with --machines: 'a,b' = Stage 4 under F = a*L_max + b*C_max (Eq.(10)) over the "
                         "locality-threshold ladder instead of the hard locality rule")
    ap.add_argument("--planner", default="stage4", choices=["stage4", "full", "alg2"],
                    help="stage4 = the headline path (step-level placement is an input, Stage 4 on the GPU); "
                         "full = Stage 1 + Alg. 3 Stages 2-3 + Stage 4 all on the GPU inside the timed step "
                         "(--machines M then restricts relocation / replication to machines of P/M ranks); "
                         "alg2 = Alg. 1 + Alg. 2 Stages 2-4 (swaps, replica search, Stage 4 under --objective a,b "
                         "over --machines M) on the GPU inside the timed step")
    ap.add_argument("--streams", type=int, default=1,
                    help="> 1: interleave the independent instances over that many CUDA streams")
    ap.add_argument("--mb-per-call", type=int, default=1,
                    help="diagnostic: one dispatch / combine call per this many consecutive micro-steps of a layer "
                         "(ranged calls); per-launch time against size separates the fixed cost of a launch from its rate")
    ap.add_argument("--strict-order", action="store_true",
                    help="do not set FOREMOE_FLAG_PLAN_STABLE: the data-path kernels then read nothing, not even "
                         "the plan arrays, before the preceding kernel of the stream has completed")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="skip the records of configs 1, 3, 5 and the config-4 size sweep that the default "
                         "(config 2, 1 GPU) run appends under other_configs after the headline's legs")
    ap.add_argument("--no-cpu-all-cores", action="store_true",
                    help="skip the all-cores leg of cpu_baseline (one oracle process per host core)")
    ap.add_argument("--tune", default="",
                    help="sweeps only: comma-separated key=value launch parameters (csrc/foremoe_data.cuh "
                         "DataTuning); loads the -DFOREMOE_TUNING build (python -m paper_2606_11867_b200.build "
                         "--tuning) instead of the product library and marks the line as a sweep")
    args = ap.parse_args()
    if args.tune:
        apply_tuning(args.tune)
    cfg = synth.config(args.config, mb_samples=args.mb_samples)
    if args.layers:
        cfg = cfg.scaled(L=args.layers)
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
