"""The paper's random-normal sweeps (Fig. 4): x ~ N(0, I_D), N = 10,000 samples quantised with a codebook of
size K by standard K-means (KM) and by GSKM; MSE, gain error, cosine similarity and the shrinkage ratio (:85).
(a-c) dimension sweep at K = 2048, (d-f) capacity sweep at D = 256.  The figure's values are not in the paper's text (and its
panel titles are garbled): only the stated trend can be compared.  Everything runs in libgsrq
(gsrq_cluster_fit / gsrq_cluster_assign / gsrq_cluster_metrics); this script only draws the samples and prints the table.

  python -m paper_2607_01065_b200.fig4_sweep [--iters 25] [--N 10000]
"""
from __future__ import annotations

import argparse
import json

import torch

from . import binding as B

D_SWEEP = [(D, 2048) for D in (8, 16, 32, 64, 128, 256)]       # (a-c): vary D, K = 2048
K_SWEEP = [(256, K) for K in (16, 64, 256, 1024, 2048, 4096)]  # (d-f): vary K, D = 256


def run_one(x: torch.Tensor, K: int, iters: int, method: int, seed: int = 0) -> dict:
    N, d = x.shape
    shapes = torch.zeros(K, d, device="cuda"); gains = torch.zeros(K, device="cuda")
    idx = torch.zeros(N, dtype=torch.int16, device="cuda")
    ws = B.cluster_workspace(N, d, K)
    st = B.gsrq_cluster_fit(x, None, K, iters, seed, method, shapes, gains, idx, ws)
    B.gsrq_cluster_assign(x, K, method, shapes, gains, idx)
    m = B.gsrq_cluster_metrics(x, K, method, shapes, gains, idx, ws)
    m["iters_run"] = st[0].iters_run
    return m


def sweep(settings=None, iters: int = 25, N: int = 10000, seed: int = 2024):
    settings = D_SWEEP + K_SWEEP if settings is None else settings
    out = []
    for D, K in settings:
        gen = torch.Generator(device="cuda"); gen.manual_seed(seed + D)
        x = torch.randn(N, D, device="cuda", generator=gen)
        out.append(dict(D=D, K=K, km=run_one(x, K, iters, 1), gskm=run_one(x, K, iters, 0)))
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--iters", type=int, default=25)
    ap.add_argument("--N", type=int, default=10000)
    a = ap.parse_args()
    print(f"{'D':>4} {'K':>5} | {'MSE km':>9} {'gskm':>9} | {'gain err km':>11} {'gskm':>9} | {'cosine km':>9} {'gskm':>7} | {'shrink km':>9} {'gskm':>6}")
    for r in sweep(iters=a.iters, N=a.N):
        k, g = r["km"], r["gskm"]
        print(f"{r['D']:>4} {r['K']:>5} | {k['mse']:9.4f} {g['mse']:9.4f} | {k['gain_err']:11.4f} {g['gain_err']:9.4f} | "
              f"{k['cosine']:9.4f} {g['cosine']:7.4f} | {k['shrinkage']:9.4f} {g['shrinkage']:6.4f}")
        print(json.dumps(r))


if __name__ == "__main__":
    main()
