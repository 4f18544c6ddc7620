"""Seeded synthetic inputs shaped like the paper's long-context workloads.

This module serves BOTH the CUDA path and the CPU oracle (tests, bench) and holds none
of the method's arithmetic: it only draws Q/K/V and plants heavy hitters.  The paper
measures on lm-eval-harness / LongBench prompts through LLaMA-2-7B;
neither weights nor datasets exist on the build or GPU boxes, so these tensors stand in
for the per-layer Q/K/V of such a prefill.

Recipe (per layer; data seed = 1000*config_id + layer):
  * Q [B,Hq,P,d], K,V [B,Hkv,L,d] ~ i.i.d. N(0,1) in fp32.
  * heavy hitters, per (batch, kv head) independently: n_h = round(rate*L) distinct
    positions uniform in [n_sink, L-n_recent); u = unit vector along the mean of the
    group's G*P proxy queries; K[b,hk,j,:] += alpha*sqrt(d)*u at those positions, i.e. a
    boost of alpha*(q.u) in logit units (emulates the paper's "pivotal tokens",
    PAPER.md:344).
  * cast to bf16 (round-to-nearest-even) unless the config is fp32.  V is payload only.
The same bytes feed both sides: generate once on one device, copy for the other.
"""
from __future__ import annotations

import math

import torch

from .configs import EvictConfig


def make_layer_inputs(cfg: EvictConfig, layer: int = 0, device="cpu"):
    """Returns (K, V, Q, planted) with planted = int64 [B,Hkv,n_h] heavy-hitter positions."""
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(cfg.data_seed(layer))
    B, Hq, Hkv, L, d, P, G = cfg.batch, cfg.Hq, cfg.Hkv, cfg.L, cfg.d, cfg.P, cfg.G
    Q = torch.randn(B, Hq, P, d, generator=gen, device=dev, dtype=torch.float32)
    K = torch.randn(B, Hkv, L, d, generator=gen, device=dev, dtype=torch.float32)
    V = torch.randn(B, Hkv, L, d, generator=gen, device=dev, dtype=torch.float32)

    n_h = int(round(cfg.hh_rate * L))
    free = L - cfg.n_sink - cfg.n_recent
    n_h = max(0, min(n_h, free))
    planted = torch.empty(B, Hkv, n_h, dtype=torch.int64, device=dev)
    if n_h > 0:
        # mean proxy-query direction of each GQA group, fp32, before any cast
        mean_q = Q.view(B, Hkv, G * P, d).mean(dim=2)
        u = mean_q / mean_q.norm(dim=-1, keepdim=True).clamp_min(1e-20)
        boost = (cfg.hh_alpha * math.sqrt(d)) * u  # [B,Hkv,d]
        for b in range(B):
            for hk in range(Hkv):
                pos = torch.randperm(free, generator=gen, device=dev)[:n_h] + cfg.n_sink
                pos, _ = torch.sort(pos)
                planted[b, hk] = pos
                K[b, hk, pos] += boost[b, hk]
    if cfg.dtype == "bf16":
        Q, K, V = Q.to(torch.bfloat16), K.to(torch.bfloat16), V.to(torch.bfloat16)
    return K.contiguous(), V.contiguous(), Q.contiguous(), planted


def make_random_inputs(B, L, Hq, Hkv, d, P, dtype="f32", seed=0, device="cpu", scale=1.0):
    """Plain N(0, scale^2) Q/K/V for small parity / property cases."""
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(seed)
    Q = torch.randn(B, Hq, P, d, generator=gen, device=dev) * scale
    K = torch.randn(B, Hkv, L, d, generator=gen, device=dev) * scale
    V = torch.randn(B, Hkv, L, d, generator=gen, device=dev)
    if dtype == "bf16":
        Q, K, V = Q.to(torch.bfloat16), K.to(torch.bfloat16), V.to(torch.bfloat16)
    return K.contiguous(), V.contiguous(), Q.contiguous()
