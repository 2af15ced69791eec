"""Seeded synthetic inputs: routing traces, micro-step boundaries, placements, activations.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA path
(``paper_2606_11867_b200.binding``).  It holds none of the method's arithmetic: it only
draws the inputs that ForeMoE's planner and dispatch consume, with the shapes and statistics
of the paper's workloads (the recipe is restated in DESIGN.md section 4):

* the routing trace the *Routing Collector* records at rollout (section 5): top-K
  expert ids per token per MoE layer, plus fp32 gate weights (BASELINE.json ``north_star``);
* micro-step boundaries ``mb_off`` (section 2.3: sequences are split into
  micro-batches processed sequentially in micro-steps);
* a step-level placement with replica slots (input to Stage 4, section 8.2),
  produced host-side by a capacity-limited LPT base placement (the M=1 reduction of
  Alg. 1) plus a step-level greedy replication;
* token activations ``x``.

The routing recorded on DAPO-Math-17k / CodeForces rollouts is not in this
container; these traces stand in for it (stable-but-skewed step-level popularity = Zipf,
micro-step volatility = per-sample Dirichlet perturbation, section 3).

The same generated arrays are handed to both sides, so parity never depends on the RNG being
reproducible across devices: generation on ``cuda`` and on ``cpu`` gives different (equally
valid) traces for the same seed.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional

import numpy as np
import torch

ACT_BF16 = 0
ACT_FP32 = 1


@dataclasses.dataclass
class TraceConfig:
    name: str
    cfg_id: int
    L: int                      # MoE layers
    E: int                      # experts
    K: int                      # top-k
    P: int                      # logical EP ranks
    Nb: int                     # base slots per rank (= E / P)
    Nr: int                     # redundant slots per rank
    H: int                      # hidden size
    act_dtype: int              # ACT_BF16 / ACT_FP32
    zipf_s: float               # per-layer popularity exponent
    dirichlet_alpha: Optional[float]   # per-(sample, layer) perturbation; None = absent
    beta: float                 # strength of the perturbation
    sample_len: List[int]       # tokens per sample
    mb_samples: int             # samples per micro-step
    max_hosts: int = 0          # cap on hosts per expert in the placement (0 = P)
    w_from_noise: bool = False  # cfg 5: gate weights = softmax over the N(0,1) part only
    seed: int = 0

    @property
    def Ns(self) -> int:
        return self.Nb + self.Nr

    @property
    def S(self) -> int:
        return self.P * self.Ns

    @property
    def T(self) -> int:
        return int(sum(self.sample_len))

    @property
    def n_mb(self) -> int:
        return (len(self.sample_len) + self.mb_samples - 1) // self.mb_samples

    def mb_off(self) -> np.ndarray:
        """Micro-step token boundaries: contiguous, sample-aligned, packed (no padding)."""
        off = [0]
        n = len(self.sample_len)
        for i in range(0, n, self.mb_samples):
            off.append(off[-1] + int(sum(self.sample_len[i:i + self.mb_samples])))
        return np.asarray(off, dtype=np.int32)

    def sample_off(self) -> np.ndarray:
        return np.concatenate([[0], np.cumsum(self.sample_len)]).astype(np.int64)

    def scaled(self, L: Optional[int] = None, n_samples: Optional[int] = None,
               sample_len: Optional[int] = None, H: Optional[int] = None,
               mb_samples: Optional[int] = None) -> "TraceConfig":
        """A reduced copy (fewer layers / samples / shorter samples / narrower rows) for tests."""
        c = dataclasses.replace(self)
        if L is not None:
            c.L = L
        lens = list(self.sample_len)
        if n_samples is not None:
            lens = lens[:n_samples]
        if sample_len is not None:
            lens = [min(x, sample_len) for x in lens]
        c.sample_len = lens
        if H is not None:
            c.H = H
        if mb_samples is not None:
            c.mb_samples = mb_samples
        c.name = self.name + "-scaled"
        return c


def lognormal_lengths(n: int, seed: int) -> List[int]:
    """Response lengths of config 4: lognormal(median 1500, sigma 0.6) clipped to [256, 8192]."""
    rng = np.random.default_rng(np.random.SeedSequence([seed, 4, 0xA11CE]))
    v = rng.lognormal(mean=math.log(1500.0), sigma=0.6, size=n)
    return [int(x) for x in np.rint(np.clip(v, 256, 8192))]


def config(cfg_id: int, mb_samples: Optional[int] = None, seed: int = 0) -> TraceConfig:
    """The five BASELINE.json configs (values the JSON leaves open follow SURVEY.md section 8)."""
    if cfg_id == 1:    # Tiny
        return TraceConfig("tiny", 1, L=1, E=8, K=2, P=4, Nb=2, Nr=1, H=256, act_dtype=ACT_FP32,
                           zipf_s=1.0, dirichlet_alpha=None, beta=0.0,
                           sample_len=[512] * 8, mb_samples=1, seed=seed)
    if cfg_id == 2:    # Qwen3-30B-A3B-shaped
        return TraceConfig("qwen3-30b-a3b", 2, L=48, E=128, K=8, P=8, Nb=16, Nr=2, H=2048,
                           act_dtype=ACT_BF16, zipf_s=1.2, dirichlet_alpha=0.3, beta=0.5,
                           sample_len=[2048] * 256, mb_samples=8, seed=seed)
    if cfg_id == 3:    # DeepSeek-V3-shaped
        return TraceConfig("deepseek-v3", 3, L=58, E=256, K=8, P=64, Nb=4, Nr=1, H=7168,
                           act_dtype=ACT_BF16, zipf_s=1.1, dirichlet_alpha=0.3, beta=0.5,
                           sample_len=[4096] * 128, mb_samples=4, seed=seed)
    if cfg_id == 4:    # micro-step size sweep (mb_samples in {1,2,4,...,64})
        return TraceConfig("mb-size-sweep", 4, L=4, E=128, K=8, P=8, Nb=16, Nr=2, H=2048,
                           act_dtype=ACT_BF16, zipf_s=1.2, dirichlet_alpha=0.3, beta=0.5,
                           sample_len=lognormal_lengths(256, seed),
                           mb_samples=mb_samples or 8, seed=seed)
    if cfg_id == 5:    # skew stress
        return TraceConfig("skew-stress", 5, L=4, E=512, K=10, P=32, Nb=16, Nr=4, H=4096,
                           act_dtype=ACT_BF16, zipf_s=2.0, dirichlet_alpha=None, beta=0.0,
                           sample_len=[32768] * 16, mb_samples=1, max_hosts=8,
                           w_from_noise=True, seed=seed)
    raise ValueError(f"unknown config {cfg_id}")


def _layer_log_popularity(cfg: TraceConfig, layer: int) -> np.ndarray:
    """log p_l[e], p_l[e] ~ rank^(-s), ranks assigned by a per-layer permutation of expert ids."""
    rng = np.random.default_rng(np.random.SeedSequence([cfg.seed, cfg.cfg_id, layer, 1]))
    perm = rng.permutation(cfg.E)
    p = np.empty(cfg.E, dtype=np.float64)
    p[perm] = (np.arange(cfg.E, dtype=np.float64) + 1.0) ** (-cfg.zipf_s)
    p /= p.sum()
    return np.log(p)


def _sample_bias(cfg: TraceConfig, layer: int) -> Optional[np.ndarray]:
    """beta * log(E * d + 1e-3), d ~ Dirichlet(alpha 1_E) per (sample, layer); [n_samples, E]."""
    if cfg.dirichlet_alpha is None:
        return None
    rng = np.random.default_rng(np.random.SeedSequence([cfg.seed, cfg.cfg_id, layer, 2]))
    d = rng.dirichlet(np.full(cfg.E, cfg.dirichlet_alpha), size=len(cfg.sample_len))
    return cfg.beta * np.log(cfg.E * d + 1e-3)


def gen_trace(cfg: TraceConfig, device: str = "cpu", chunk_tokens: int = 65536):
    """Routing trace of one RL step.

    Returns ``ids`` int32 [L, T, K] (top-K in descending-logit order), ``w`` fp32 [L, T, K]
    (softmax renormalised over the K selected logits) and ``mb_off`` int32 [n_mb + 1], all on
    ``device``.  logit[t][e] = log p_l[e] + beta*log(E*d_{sample(t),l}[e] + 1e-3) + N(0,1).
    """
    dev = torch.device(device)
    L, T, K, E = cfg.L, cfg.T, cfg.K, cfg.E
    ids = torch.empty((L, T, K), dtype=torch.int32, device=dev)
    w = torch.empty((L, T, K), dtype=torch.float32, device=dev)
    samp_off = cfg.sample_off()
    sample_of_token = torch.from_numpy(
        np.repeat(np.arange(len(cfg.sample_len), dtype=np.int64), cfg.sample_len)).to(dev)
    for l in range(L):
        logp = torch.from_numpy(_layer_log_popularity(cfg, l)).to(dev, torch.float32)
        bias = _sample_bias(cfg, l)
        bias_t = None if bias is None else torch.from_numpy(bias).to(dev, torch.float32)
        gen = torch.Generator(device=dev)
        gen.manual_seed((cfg.seed * 1000003 + cfg.cfg_id * 7919 + l) & 0x7FFFFFFF)
        for t0 in range(0, T, chunk_tokens):
            t1 = min(T, t0 + chunk_tokens)
            noise = torch.randn((t1 - t0, E), generator=gen, device=dev, dtype=torch.float32)
            logit = noise + logp[None, :]
            if bias_t is not None:
                logit = logit + bias_t[sample_of_token[t0:t1]]
            top_v, top_i = torch.topk(logit, K, dim=1, largest=True, sorted=True)
            if cfg.w_from_noise:
                top_v = torch.gather(noise, 1, top_i)
            ids[l, t0:t1] = top_i.to(torch.int32)
            w[l, t0:t1] = torch.softmax(top_v, dim=1)
    del samp_off
    mb_off = torch.from_numpy(cfg.mb_off()).to(dev)
    return ids, w, mb_off


def gen_activations(cfg: TraceConfig, n_tokens: int, tag: int, device: str = "cpu") -> torch.Tensor:
    """x[n_tokens, H] ~ N(0,1), rounded to bf16 (fp32 in config 1)."""
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed((cfg.seed * 1000003 + cfg.cfg_id * 7919 + 0x5EED + tag) & 0x7FFFFFFF)
    x = torch.randn((n_tokens, cfg.H), generator=gen, device=dev, dtype=torch.float32)
    if cfg.act_dtype == ACT_BF16:
        return x.to(torch.bfloat16)
    return x


def gen_placement(cfg: TraceConfig, step_hist: np.ndarray) -> np.ndarray:
    """Step-level placement ``slot_expert`` int32 [L, S] (global slot j = rank*Ns + local).

    Base: experts in descending step total, each to the least-loaded rank that still has a free
    base slot (Alg. 1 rank-level LPT, with the N_b capacity).  Replicas: P*N_r
    rounds, each giving the expert with the largest step_total / copies a redundant slot on the
    least-loaded rank that has a free redundant slot and does not host it yet.  This is input
    preparation (the harness-side stand-in for Stages 1-3), not part of the measured path.
    """
    L, E, P, Nb, Nr, Ns = cfg.L, cfg.E, cfg.P, cfg.Nb, cfg.Nr, cfg.Ns
    assert Nb * P == E
    max_hosts = cfg.max_hosts or P
    out = np.full((L, P * Ns), -1, dtype=np.int32)
    for l in range(L):
        tot = step_hist[l].astype(np.float64)
        order = sorted(range(E), key=lambda e: (-tot[e], e))
        rank_load = np.zeros(P)
        nbase = np.zeros(P, dtype=np.int64)
        hosts = [[] for _ in range(E)]          # ranks hosting e
        for e in order:
            cand = [r for r in range(P) if nbase[r] < Nb]
            r = min(cand, key=lambda r: (rank_load[r], r))
            out[l, r * Ns + nbase[r]] = e
            nbase[r] += 1
            rank_load[r] += tot[e]
            hosts[e].append(r)
        nred = np.zeros(P, dtype=np.int64)
        copies = np.ones(E)
        for _ in range(P * Nr):
            share = tot / copies
            load = np.zeros(P)
            for e in range(E):
                for r in hosts[e]:
                    load[r] += share[e]
            placed = False
            for e in sorted(range(E), key=lambda e: (-share[e], e)):
                if len(hosts[e]) >= max_hosts or share[e] <= 0:
                    continue
                cand = [r for r in range(P) if nred[r] < Nr and r not in hosts[e]]
                if not cand:
                    continue
                r = min(cand, key=lambda r: (load[r], r))
                out[l, r * Ns + Nb + nred[r]] = e
                nred[r] += 1
                hosts[e].append(r)
                copies[e] += 1
                placed = True
                break
            if not placed:
                break
    return out


def gen_tok_src(cfg: TraceConfig) -> np.ndarray:
    """Source rank of every token (int32 [T]) for the per-source Stage 4:
    every micro-step's token range is cut into P contiguous, near-equal shares, share s held by
    logical rank s -- each EP rank contributes its part of the micro-batch to the dispatch
    ("source rank s")."""
    off = cfg.mb_off().astype(np.int64)
    out = np.empty(cfg.T, dtype=np.int32)
    for i in range(cfg.n_mb):
        a, b = int(off[i]), int(off[i + 1])
        if b > a:
            out[a:b] = (np.arange(b - a, dtype=np.int64) * cfg.P // (b - a)).astype(np.int32)
    return out


def natural_placement(cfg: TraceConfig) -> np.ndarray:
    """The un-balanced default: expert e on rank e // Nb, no replicas (redundant slots empty)."""
    out = np.full((cfg.L, cfg.S), -1, dtype=np.int32)
    for e in range(cfg.E):
        r, b = divmod(e, cfg.Nb)
        out[:, r * cfg.Ns + b] = e
    return out
