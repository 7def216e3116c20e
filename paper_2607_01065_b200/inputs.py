"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is shared by the tests, bench.py and the oracle-vs-CUDA parity harness.  It
holds NONE of the method's arithmetic: only random draws shaped like the paper's
workloads (LLaMA-3-8B KV: 8 KV heads x head_dim 128), the bf16 storage
cast, and the seeded fit-token sample of config 4.  These tensors STAND IN for the real
WikiText-2 / C4 / SlimPajama activations the paper measures on (PAPER.md:214, :246,
:252), which do not exist here.

Recipe (numpy default_rng(seed), draws in the order listed, float64 then cast):
  data seed = 1000 + 10*cfg + {0: K-like, 1: V-like, 2: weights, 3: fit sample}.
  K-like: Z~N(0,1); 4 outlier channels per head (rng.choice(128,4,replace=False)) x10;
          per-channel scale exp(0.3*N(0,1)) [128]; cast RN-even to bf16.
  V-like: Z~Student-t(nu=4); per-token factor exp(0.5*N(0,1)) shared by heads; bf16.
  weights: exp(N(0,1)) per token, divided by the mean (heavy-tailed saliency).
  cfg 0:  [4096, 8] fp32, Z*exp(0.5*N(0,1)) per row, uniform weights.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
import torch

HEADS, HEAD_DIM = 8, 128


@dataclass(frozen=True)
class Config:
    cfg: int
    name: str
    G: int
    T: int
    hd: int
    d: int
    K: int
    S: int
    iters: int
    dtype: str            # "f32" | "bf16"
    kinds: tuple          # which tensors the config has: ("k",), ("v",), ("k","v")
    n_fit_tokens: int = 0  # 0 = fit on all tokens
    head_inner: bool = False  # memory layout [T][G][hd] instead of [G][T][hd]


CONFIGS = {
    0: Config(0, "tiny-sanity", 1, 4096, 8, 8, 16, 2, 10, "f32", ("x",)),
    1: Config(1, "k-cache-8x4096x128", HEADS, 4096, HEAD_DIM, 16, 256, 2, 20, "bf16", ("k",)),
    2: Config(2, "v-cache-8x16384x128", HEADS, 16384, HEAD_DIM, 16, 256, 1, 20, "bf16", ("v",)),
    3: Config(3, "bitrate-sweep-8x32768x128", HEADS, 32768, HEAD_DIM, 16, 256, 4, 20, "bf16", ("k", "v")),
    4: Config(4, "long-context-8x131072x8x128", HEADS, 8 * 131072, HEAD_DIM, 16, 256, 2, 10, "bf16",
              ("k", "v"), n_fit_tokens=65536, head_inner=True),
}


def bf16_round(x: np.ndarray) -> np.ndarray:
    """fp32/fp64 -> nearest-even bf16, returned as the exact fp32 values."""
    t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32))
    return t.to(torch.bfloat16).to(torch.float32).numpy()


def seed_of(cfg: int, what: str) -> int:
    return 1000 + 10 * cfg + {"k": 0, "x": 0, "v": 1, "w": 2, "fit": 3}[what]


def k_like(G: int, T: int, hd: int, seed: int) -> np.ndarray:
    """[G][T][hd] key-like tensor: outlier channels + per-channel scale (bf16-exact fp32)."""
    rng = np.random.default_rng(seed)
    out = np.empty((G, T, hd), dtype=np.float32)
    for g in range(G):
        z = rng.standard_normal((T, hd))
        ch = rng.choice(hd, 4, replace=False)
        scale = np.exp(0.3 * rng.standard_normal(hd))
        z[:, ch] *= 10.0
        out[g] = bf16_round(z * scale[None, :])
    return out


def v_like(G: int, T: int, hd: int, seed: int) -> np.ndarray:
    """[G][T][hd] value-like tensor: Student-t(4) entries x per-token lognormal(0,0.5) factor."""
    rng = np.random.default_rng(seed)
    tok = np.exp(0.5 * rng.standard_normal(T))
    out = np.empty((G, T, hd), dtype=np.float32)
    for g in range(G):
        z = rng.standard_t(4.0, size=(T, hd))
        out[g] = bf16_round(z * tok[:, None])
    return out


def tiny(seed: int, N: int = 4096, d: int = 8) -> np.ndarray:
    """cfg 0: [1][N][d] fp32, N(0,1) rows scaled by lognormal(0,0.5)."""
    rng = np.random.default_rng(seed)
    z = rng.standard_normal((N, d))
    f = np.exp(0.5 * rng.standard_normal(N))
    return (z * f[:, None]).astype(np.float32)[None]


def token_weights(T: int, seed: int) -> np.ndarray:
    """[T] lognormal(0,1) saliency weights normalised to mean 1 (fp32)."""
    rng = np.random.default_rng(seed)
    w = np.exp(rng.standard_normal(T))
    return (w / w.mean()).astype(np.float32)


def fit_sample(G: int, T: int, n: int, seed: int) -> np.ndarray:
    """[G][n] sorted distinct token ids per head (cfg 4's seeded fit sample, reading c-S)."""
    rng = np.random.default_rng(seed)
    return np.stack([np.sort(rng.choice(T, n, replace=False)) for _ in range(G)]).astype(np.int64)


def make(cfg: int, kind: str | None = None, T: int | None = None):
    """Inputs of a config (optionally shortened to T tokens for CPU-sized parity cases).

    Returns dict(x [G][T][hd] fp32 values, w [T] fp32 or None, fit_tokens [G][n] or None, config).
    """
    c = CONFIGS[cfg]
    T = c.T if T is None else T
    kind = c.kinds[0] if kind is None else kind
    if cfg == 0:
        x = tiny(seed_of(0, "x"), T, c.d)
        w = None
    else:
        gen = k_like if kind == "k" else v_like
        x = gen(c.G, T, c.hd, seed_of(cfg, kind))
        w = token_weights(T, seed_of(cfg, "w"))
    fit = None
    if c.n_fit_tokens:
        n = min(c.n_fit_tokens, max(T // 16, 1))
        fit = fit_sample(c.G, T, n, seed_of(cfg, "fit"))
    return dict(x=x, w=w, fit_tokens=fit, config=c, kind=kind, T=T)


def cfg4_device(kind: str = "k", T: int = 8 * 131072, n_fit: int = 65536, G: int = HEADS, hd: int = HEAD_DIM,
                device: str = "cuda", chunk: int = 131072, seed: int | None = None):
    """BASELINE config 4 drawn ON THE DEVICE (a 2.1 GB tensor is too slow to draw with numpy): head-inner layout
    [T][G][hd] bf16, per-token weights [T] fp32 (lognormal(0,1) / mean) and the sorted seeded fit sample [G][n_fit]
    int64.  Same recipes as k_like / v_like / token_weights / fit_sample with a seeded torch CUDA generator
    (seed_of(4, kind) unless `seed` is given); draws in the order: per-head statistics, tensor chunks, weights, fit sample.  The oracle is
    given copies of the same bits (tests copy the rows they need to the host).
      k: N(0,1) x per-channel scale exp(0.3 N(0,1)), 4 outlier channels per head x10 (fixed over batch and tokens).
      v: Student-t(nu=4) = N(0,1) / sqrt(chi2_4 / 4), x per-(batch, token) factor exp(0.5 N(0,1)) shared by heads."""
    gen = torch.Generator(device=device)
    gen.manual_seed(seed_of(4, kind) if seed is None else seed)
    x = torch.empty(T, G, hd, dtype=torch.bfloat16, device=device)
    if kind == "k":
        scale = torch.exp(0.3 * torch.randn(G, hd, device=device, generator=gen))
        for g in range(G):
            scale[g, torch.randperm(hd, device=device, generator=gen)[:4]] *= 10.0
        for t0 in range(0, T, chunk):
            n = min(chunk, T - t0)
            x[t0:t0 + n] = (torch.randn(n, G, hd, device=device, generator=gen) * scale).to(torch.bfloat16)
    else:
        for t0 in range(0, T, chunk):
            n = min(chunk, T - t0)
            z = torch.randn(n, G, hd, device=device, generator=gen)
            chi = torch.zeros(n, G, hd, device=device)
            for _ in range(4):
                chi += torch.randn(n, G, hd, device=device, generator=gen) ** 2
            tok = torch.exp(0.5 * torch.randn(n, 1, 1, device=device, generator=gen))
            x[t0:t0 + n] = (z / torch.sqrt(chi / 4.0) * tok).to(torch.bfloat16)
            del z, chi
    w = torch.exp(torch.randn(T, device=device, generator=gen))
    w /= w.mean()
    fit = torch.stack([torch.sort(torch.randperm(T, device=device, generator=gen)[:n_fit]).values
                       for _ in range(G)]).contiguous()
    return dict(x=x, w=w, fit_tokens=fit)
