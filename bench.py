#!/usr/bin/env python
"""bench.py -- one JSON line per run (see DESIGN.md section 7 for what each key means).

A "step" is one pass of the whole hot path over one synthetic layer tensor of BASELINE.json
config 1 (8 KV heads x 4096 tokens x 128, bf16, d=16, K=256, S=2, 20 iterations/stage):
for each stage s: gsrq_fit_stage(s) -> fused gsrq_encode of stages [0, s] (its residual feeds the
next fit; the last one is the final encode); then gsrq_decode.
value = KV vectors (token x head) through the whole step per second, summed over ranks.
Unless --no-big, rank 0 also runs BASELINE.json config 4 (one 8 x 131072-token batch, head-inner
layout, 2.1 GB): fit on a 65,536-token sample per head, full-cache encode, full-cache decode --
the sizes at which "fraction of the HBM / tensor roofline" is physically meaningful.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--cfg 1|2] [--no-big]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np
import torch

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2607_01065_b200 import inputs  # noqa: E402

METRIC = "gsrq_fit_encode_decode_kv_vectors_per_s"
UNIT = "KV vectors/s"


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return dict(hbm_gbs=d["hbm_gbs"], bf16_tflops=d["bf16_tflops"], bf16_tflops_sustained=d["bf16_tflops_sustained"],
                    source="MEASURED_PEAKS.json")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback (B200_PROFILING.md)")


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks / throttle reasons every 20 ms while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.stop_flag, self.proc = index, [], False, None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE, text=True)
            for line in self.proc.stdout:
                self.samples.append((time.perf_counter(), [t.strip() for t in line.split(",")]))
                if self.stop_flag:
                    break
        except Exception:
            pass

    def finish(self, t0=None, t1=None):
        """Median SM clock and throttle reasons over the samples taken in [t0, t1] (all samples if none fall inside)."""
        self.stop_flag = True
        if self.proc:
            self.proc.terminate()
        inside = [f for (t, f) in self.samples if t0 is not None and t0 <= t <= t1]
        rows = inside if inside else [f for (_, f) in self.samples]
        sm = [float(r[0]) for r in rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in rows if len(r) >= 6 for i in range(4) if r[2 + i].lower().startswith("active")})
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None, reasons=reasons,
                    samples=len(sm), samples_in_timed_region=len(inside))


def oracle_step(x, w, c):
    """The CPU oracle doing the same step (fit + encode every stage, then decode)."""
    from oracle import gsrq_oracle as o
    out = o.gsrq_fit_encode(x, w, c.d, c.K, c.S, c.iters, seed=0)
    o.decode(out["codes"], out["shapes"], out["gains"], c.hd, bf16=(c.dtype == "bf16"))
    return out


def run_reference(args, c):
    """--impl reference: the oracle as it stands on the host cores, same config / metric."""
    from oracle import gsrq_oracle as o
    o.build()
    dd = inputs.make(c.cfg)
    x, w = dd["x"], dd["w"]
    for _ in range(min(args.warmup, 1)):
        oracle_step(x[:1], w, c)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_step(x, w, c)
    dt = (time.perf_counter() - t0) / args.steps
    val = c.G * c.T / dt
    line = dict(metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=dt * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", impl="reference",
                config=dict(workload=f"cfg{c.cfg}:{c.name}", G=c.G, T=c.T, hd=c.hd, d=c.d, K=c.K, S=c.S, iters=c.iters),
                cpu_baseline=dict(value=val, unit=UNIT, cores=o.n_threads(), kind="oracle",
                                  sample=f"whole cfg{c.cfg} step (all {c.G} heads), {args.steps} step(s)"),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


def rank_seed(cfg: int, what: str, rank: int) -> int:
    """Replicas: rank r works on its own synthetic layer; rank 0 uses the documented seeds."""
    return inputs.seed_of(cfg, what) + 100 * rank


def whole_job_value(local_seconds: float, units_per_rank: float, world: int, device) -> tuple:
    """Weak scaling without a data-path collective: every rank processes units_per_rank units; the job takes as
    long as its slowest rank (MAX over ranks of the device-timed duration).  Returns (value, max_seconds)."""
    t = torch.tensor([local_seconds], device=device, dtype=torch.float64)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    mx = float(t.item())
    return world * units_per_rank / mx, mx


def run_cfg4(B, pk):
    """BASELINE.json config 4 for one tensor (K-like): batch 8 x 131072 tokens x 8 KV heads x 128, bf16, head-inner
    layout [B*T][G][hd] (2.147 GB); d=16, K=256, S=2, 10 iterations; codebooks fitted on a seeded 65,536-token
    sample per head, then full-cache encode and decode.  Same generator recipe as inputs.k_like, drawn on the
    device with a seeded torch generator."""
    c = inputs.CONFIGS[4]
    G, hd, d, K, S, iters = c.G, c.hd, c.d, c.K, c.S, c.iters
    T, n_fit, M = 8 * 131072, 65536, hd // d
    gen = torch.Generator(device="cuda")
    gen.manual_seed(inputs.seed_of(4, "k"))
    scale = torch.exp(0.3 * torch.randn(G, hd, device="cuda", generator=gen))
    for g in range(G):
        scale[g, torch.randperm(hd, device="cuda", generator=gen)[:4]] *= 10.0
    x = torch.empty(T, G, hd, dtype=torch.bfloat16, device="cuda")
    for t0 in range(0, T, 131072):
        x[t0:t0 + 131072] = (torch.randn(131072, G, hd, device="cuda", generator=gen) * scale).to(torch.bfloat16)
    w = torch.exp(torch.randn(T, device="cuda", generator=gen))
    w /= w.mean()
    fit = torch.stack([torch.sort(torch.randperm(T, device="cuda", generator=gen)[:n_fit]).values for _ in range(G)]).contiguous()
    view = B.view_of(x, d, head_inner=True)
    shapes = torch.zeros(G, S, K, d, device="cuda")
    gains = torch.zeros(G, S, K, device="cuda")
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, S, n_fit)
    codes = torch.zeros(S, G, T * M, dtype=torch.uint8, device="cuda")
    out = torch.empty_like(x)

    def timed(f, n=3):
        ts = []
        for _ in range(n):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); f(); b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return float(np.median(ts))

    def fit_all():
        for s in range(S):   # residual re-derived from kv + earlier stages on the fit rows
            B.gsrq_fit_stage(x, view, w, 0, fit, cb, s, None, iters, 0, ws, want_stats=False)

    fit_all()
    fit_ms = timed(fit_all, 2)
    enc = lambda: B.gsrq_encode(x, view, cb, 0, S, codes, None, ws)
    enc()
    enc_ms = timed(enc)
    B.gsrq_profile_enable(True)
    enc()
    torch.cuda.synchronize()
    pr = B.gsrq_profile_read()
    B.gsrq_profile_enable(False)
    dec = lambda: B.gsrq_decode(codes, cb, S, out, view)
    dec()
    dec_ms = timed(dec, 5)
    rows = G * T * M
    enc_tf = 2.0 * K * d * rows * S / (enc_ms * 1e-3) / 1e12
    tc_tf = 2.0 * K * d * rows * S / (pr["encode"][0] * 1e-3) / 1e12 if pr["encode"][0] > 0 else None
    dec_bytes = rows * S + rows * 2 * d
    dec_gbs = dec_bytes / (dec_ms * 1e-3) / 1e9
    # sanity: decode(encode(x)) must be closer to x than 0 is (relative residual energy < 1)
    err = float(((out[:4096].float() - x[:4096].float()) ** 2).sum() / (x[:4096].float() ** 2).sum())
    return dict(workload="cfg4:k-cache-8x131072x8x128 head-inner, fit on 65536-token sample/head", T=T, G=G, S=S, iters=iters,
                bytes=x.numel() * 2, fit_ms=fit_ms,
                encode=dict(ms=enc_ms, kv_vectors_per_s=G * T / (enc_ms * 1e-3), bound="tensor", achieved_tflops=enc_tf,
                            frac=enc_tf / pk["bf16_tflops_sustained"], tc_kernel_ms=pr["encode"][0], tc_kernel_tflops=tc_tf,
                            exact_path_ms=pr["refine"][0]),
                decode=dict(ms=dec_ms, gb_per_s=dec_gbs, bound="hbm", frac=dec_gbs / pk["hbm_gbs"], bytes=dec_bytes),
                rel_residual_energy_first_4096_tokens=err)


def run_cfg2(B, pk):
    """BASELINE.json config 2: V-like 8 x 16384 x 128 (Student-t, per-token norms), d=16, K=256, S=1, 20 iterations;
    fit + encode, and the decode of the whole layer timed (33.5 MB out: L2-resident, so GB/s is effective)."""
    c = inputs.CONFIGS[2]
    G, T, hd, d, K, S, iters = c.G, c.T, c.hd, c.d, c.K, c.S, c.iters
    M = hd // d
    x = torch.from_numpy(inputs.v_like(G, T, hd, inputs.seed_of(2, "v"))).to(torch.bfloat16).cuda()
    w = torch.from_numpy(inputs.token_weights(T, inputs.seed_of(2, "w"))).cuda()
    view = B.view_of(x, d)
    shapes = torch.zeros(G, S, K, d, device="cuda")
    gains = torch.zeros(G, S, K, device="cuda")
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, S, 0)
    codes = torch.zeros(S, G, T * M, dtype=torch.uint8, device="cuda")
    out = torch.empty_like(x)

    def timed(f, n=5):
        ts = []
        for _ in range(n):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); f(); b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return float(np.median(ts))

    fit = lambda: B.gsrq_fit_stage(x, view, w, 0, None, cb, 0, None, iters, 0, ws, want_stats=False)
    enc = lambda: B.gsrq_encode(x, view, cb, 0, S, codes, None, ws)
    dec = lambda: B.gsrq_decode(codes, cb, S, out, view)
    fit(); enc(); dec()
    fit_ms, enc_ms, dec_ms = timed(fit, 3), timed(enc), timed(dec)
    rows = G * T * M
    by = rows * S + rows * 2 * d
    return dict(workload="cfg2:v-cache-8x16384x128, S=1", fit_ms=fit_ms, encode_ms=enc_ms,
                encode_kv_vectors_per_s=G * T / (enc_ms * 1e-3),
                encode_tensor_frac=2.0 * K * d * rows * S / (enc_ms * 1e-3) / 1e12 / pk["bf16_tflops_sustained"],
                decode_ms=dec_ms, decode_gb_per_s=by / (dec_ms * 1e-3) / 1e9, decode_hbm_frac=by / (dec_ms * 1e-3) / 1e9 / pk["hbm_gbs"])


def run_cfg3(B, pk):
    """BASELINE.json config 3 for the K-like tensor (8 x 32768 x 128, bf16): one S=4 fit (20 iterations per stage),
    then encode throughput and decode GB/s for S = 1..4 (prefixes of the same codebooks) and the
    weighted distortion after each stage."""
    c = inputs.CONFIGS[3]
    G, T, hd, d, K, S, iters = c.G, c.T, c.hd, c.d, c.K, c.S, c.iters
    M = hd // d
    x = torch.from_numpy(inputs.k_like(G, T, hd, inputs.seed_of(3, "k"))).to(torch.bfloat16).cuda()
    w = torch.from_numpy(inputs.token_weights(T, inputs.seed_of(3, "w"))).cuda()
    view = B.view_of(x, d)
    shapes = torch.zeros(G, S, K, d, device="cuda")
    gains = torch.zeros(G, S, K, device="cuda")
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, S, 0)
    codes = torch.zeros(S, G, T * M, dtype=torch.uint8, device="cuda")
    residual = torch.zeros(G, T * M, d, device="cuda")
    out = torch.empty_like(x)
    w_rows = w.repeat_interleave(M).double()
    e0 = float((w_rows[None] * (x.float().reshape(G, T * M, d).double() ** 2).sum(-1)).sum())

    def fit_all(want_dist):
        dist = []
        for s in range(S):
            B.gsrq_fit_stage(x, view, w, 0, None, cb, s, residual if s else None, iters, 0, ws, want_stats=False)
            B.gsrq_encode(x, view, cb, 0, s + 1, codes, residual, ws)
            if want_dist:
                dist.append(float((w_rows[None] * (residual.double() ** 2).sum(-1)).sum()) / e0)
        return dist

    dist = fit_all(True)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(); fit_all(False); b.record()
    torch.cuda.synchronize()
    fit_ms = a.elapsed_time(b)
    rows = G * T * M
    sweep = []
    for n in range(1, S + 1):
        ts, td = [], []
        for _ in range(5):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); B.gsrq_encode(x, view, cb, 0, n, codes, None, ws); b.record()
            torch.cuda.synchronize(); ts.append(a.elapsed_time(b))
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); B.gsrq_decode(codes, cb, n, out, view); b.record()
            torch.cuda.synchronize(); td.append(a.elapsed_time(b))
        em, dm = float(np.median(ts)), float(np.median(td))
        by = rows * n + rows * 2 * d
        sweep.append(dict(S=n, bits_per_element=n * 8.0 / d, encode_ms=em, encode_kv_vectors_per_s=G * T / (em * 1e-3),
                          encode_tensor_frac=2.0 * K * d * rows * n / (em * 1e-3) / 1e12 / pk["bf16_tflops_sustained"],
                          decode_ms=dm, decode_gb_per_s=by / (dm * 1e-3) / 1e9, decode_hbm_frac=by / (dm * 1e-3) / 1e9 / pk["hbm_gbs"],
                          rel_weighted_distortion=dist[n - 1]))
    return dict(workload="cfg3:k-cache-8x32768x128, S=4 fit, prefixes S=1..4 (67 MB: L2-resident, effective GB/s)",
                fit_and_encode_ms=fit_ms, sweep=sweep)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cfg", type=int, default=1, choices=[1, 2])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-big", action="store_true", help="skip the config-4 (2.1 GB) encode / decode leg")
    ap.add_argument("--only-big", action="store_true", help="run only the config-4 leg and print its JSON (profiling aid)")
    args = ap.parse_args()
    c = inputs.CONFIGS[args.cfg]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        if rank == 0:
            run_reference(args, c)
        return

    import __graft_entry__ as ge
    from paper_2607_01065_b200 import binding as B
    if rank == 0:
        ge.build()
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist.barrier()
    torch.cuda.set_device(local)
    B.lib()
    if args.only_big:
        if rank == 0:
            print(json.dumps(dict(impl="ours", cfg4=run_cfg4(B, peaks()))))
        return

    # ---- inputs (replicas: rank r works on its own layer; rank 0 is the documented seeds) ----
    kind = c.kinds[0]
    gen = inputs.k_like if kind == "k" else inputs.v_like
    x_np = gen(c.G, c.T, c.hd, rank_seed(c.cfg, kind, rank))
    w_np = inputs.token_weights(c.T, rank_seed(c.cfg, "w", rank))
    x_host = torch.from_numpy(x_np).to(torch.bfloat16).pin_memory()
    w_host = torch.from_numpy(w_np).pin_memory()
    x = x_host.cuda()
    w = w_host.cuda()
    view = B.view_of(x, c.d)
    G, T, hd, d, K, S = c.G, c.T, c.hd, c.d, c.K, c.S
    M = hd // d
    shapes = torch.zeros(G, S, K, d, device="cuda")
    gains = torch.zeros(G, S, K, device="cuda")
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, S, 0)
    codes = torch.zeros(S, G, T * M, dtype=torch.uint8, device="cuda")
    residual = torch.zeros(G, T * M, d, device="cuda")
    out = torch.zeros_like(x)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def step():
        for s in range(S):
            B.gsrq_fit_stage(x, view, w, 0, None, cb, s, residual if s else None, c.iters, 0, ws, want_stats=False)
            B.gsrq_encode(x, view, cb, 0, s + 1, codes, residual if s + 1 < S else None, ws)
        B.gsrq_decode(codes, cb, S, out, view)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()                          # nvidia-smi takes a moment to come up: start it before the warm-up
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    t_region0 = time.perf_counter()
    l0 = B.gsrq_launch_count()
    evs = []
    for _ in range(args.steps):
        flush.fill_(1)                      # evict the previous step's data from L2 (not timed)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); step(); b.record()
        evs.append((a, b))
    barrier()
    launches = B.gsrq_launch_count() - l0
    ms = sum(a.elapsed_time(b) for a, b in evs)
    value, max_s = whole_job_value(ms * 1e-3 / args.steps, G * T, world, "cuda")
    ms_per_step = max_s * 1e3

    # ---- per-kernel device time, measured live with CUDA events around every launch ----
    B.gsrq_profile_enable(True)
    for _ in range(2):
        step()
    torch.cuda.synchronize()
    prof = B.gsrq_profile_read()
    B.gsrq_profile_enable(False)
    # decode alone (cold L2) for the decode GB/s figure
    dts = []
    for _ in range(5):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); B.gsrq_decode(codes, cb, S, out, view); b.record()
        torch.cuda.synchronize()
        dts.append(a.elapsed_time(b))
    dec_ms = float(np.median(dts))
    dec_bytes = G * T * M * S + G * T * hd * 2
    ets = []
    for _ in range(5):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); B.gsrq_encode(x, view, cb, 0, S, codes, None, ws); b.record()
        torch.cuda.synchronize()
        ets.append(a.elapsed_time(b))
    enc_ms = float(np.median(ets))
    # encode-on-append (PAPER.md:443 (i)): latency of quantising the newest token(s) of a batch of sequences
    app = []
    for n_new in (8, 16, 32):
        chunk = x[:, :n_new]
        cv = B.view_of(chunk, d)
        B.gsrq_encode_append(chunk, cv, cb, S, codes, T * M, 0)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(20):
            B.gsrq_encode_append(chunk, cv, cb, S, codes, T * M, 0)
        b.record()
        torch.cuda.synchronize()
        app.append(dict(new_tokens=n_new, us_per_call=a.elapsed_time(b) * 1e3 / 20))

    # ---- end to end through the host-buffer C-ABI call: H2D + fit + encode + decode + D2H ----
    sh_h = torch.empty(G, S, K, d).pin_memory(); ga_h = torch.empty(G, S, K).pin_memory()
    co_h = torch.empty(S, G, T * M, dtype=torch.uint8).pin_memory(); out_h = torch.empty_like(x_host).pin_memory()
    for _ in range(2):
        B.gsrq_pipeline_host(x_host, view, w_host, K, S, c.iters, 0, sh_h, ga_h, co_h, out_h)
    barrier()
    t0 = time.perf_counter()
    n_e2e = max(3, args.steps // 2)
    for _ in range(n_e2e):
        B.gsrq_pipeline_host(x_host, view, w_host, K, S, c.iters, 0, sh_h, ga_h, co_h, out_h)
    barrier()
    e2e_s = (time.perf_counter() - t0) / n_e2e
    e2e_val, _ = whole_job_value(e2e_s, G * T, world, "cuda")
    h2d = x_host.numel() * 2 + w_host.numel() * 4
    d2h = sh_h.numel() * 4 + ga_h.numel() * 4 + co_h.numel() + out_h.numel() * 2
    clocks = sampler.finish(t_region0, time.perf_counter())
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()      # no collective below: the remaining legs run on rank 0 alone

    if rank != 0:
        return
    big = sweep3 = v2 = None
    if not args.no_big:
        del flush
        torch.cuda.empty_cache()
        big = run_cfg4(B, peaks())
        torch.cuda.empty_cache()
        sweep3 = run_cfg3(B, peaks())
        torch.cuda.empty_cache()
        v2 = run_cfg2(B, peaks())
    pk = peaks()
    # Rooflines of the step's kernels, from the live CUDA-event brackets (two profiled steps).
    # Algorithmic work: scoring pass 2*K*d flops per sub-vector; update kernel one read of
    # the fp32 row + 1/(||r||+eps) + code = 4d + 9 bytes per sub-vector; decode S + 2d bytes per sub-vector.
    rows_per_launch = G * T * M
    tot_ms = sum(v[0] for v in prof.values())

    # DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the cfg-1 kernels from the ncu --set full
    # captures summarised in profiles/r1_v5_ncu_full.md; None for workloads that were not captured
    NCU_TRAFFIC = {"score": 10.09e6, "update": 21.42e6} if c.cfg == 1 else {}

    def kern(name, cls, bound, work_per_launch, peak, unit):
        ms, n = prof[cls]
        per = ms / max(n, 1)
        ach = work_per_launch / (per * 1e-3) / (1e12 if bound == "tensor" else 1e9) if per > 0 else 0.0
        return dict(bound=bound, kernel=name, achieved=ach, peak=peak, unit=unit, frac=ach / peak, traffic=NCU_TRAFFIC.get(cls),
                    algorithmic_per_launch=work_per_launch,
                    ms_per_launch=per, launches=n // 2, share_of_step=ms / tot_ms if tot_ms else None)

    kerns = [
        kern("tc::k_score_tc (tcgen05 scoring + arg-max, fit passes)", "score", "tensor", 2.0 * K * d * rows_per_launch,
             pk["bf16_tflops_sustained"], "TFLOP/s"),
        kern("k_update (segmented fp64 reduction + Eq. 7/8)", "update", "hbm", rows_per_launch * (4.0 * d + 9.0),
             pk["hbm_gbs"], "GB/s"),
        kern("tc::k_encode_tc (fused S-stage encode)", "encode", "tensor", 0.0, pk["bf16_tflops_sustained"], "TFLOP/s"),
    ]
    # the encode class mixes [0,1) and [0,2) launches: algorithmic flops of one step's encodes / their summed time
    enc_cls_ms = prof["encode"][0] / 2
    if enc_cls_ms > 0:
        ach = 2.0 * K * d * rows_per_launch * sum(range(1, S + 1)) / (enc_cls_ms * 1e-3) / 1e12
        kerns[2].update(achieved=ach, frac=ach / pk["bf16_tflops_sustained"])
    dom = max(kerns, key=lambda kk: kk["share_of_step"] or 0.0)
    roofline = dict(dom)
    roofline["peak_source"] = pk["source"] + (" (sustained bf16: kernel timed inside a long step)" if dom["bound"] == "tensor" else " (copy bandwidth)")
    roofline["by_class"] = {k: dict(ms=v[0] / 2, launches=v[1] // 2) for k, v in prof.items()}
    roofline["other_kernels"] = [kk for kk in kerns if kk is not dom]
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="bf16 in, fp32/fp64 arithmetic",
                data="synthetic", impl="ours",
                config=dict(workload=f"cfg{c.cfg}:{c.name}", G=G, T=T, hd=hd, d=d, K=K, S=S, iters=c.iters,
                            l2="flushed between steps (256 MiB write, untimed)", parallelism="replicas"),
                clocks=clocks, gpu_launches=int(launches),
                e2e=dict(value=e2e_val, unit=UNIT, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h,
                         call="gsrq_pipeline_host"),
                roofline=roofline,
                encode=dict(kv_vectors_per_s=G * T / (enc_ms * 1e-3), ms=enc_ms, stages=S,
                            tensor_frac=(2.0 * K * d * rows_per_launch * S / (enc_ms * 1e-3) / 1e12) / pk["bf16_tflops"]),
                decode=dict(gb_per_s=dec_bytes / (dec_ms * 1e-3) / 1e9, ms=dec_ms, bytes=dec_bytes,
                            hbm_frac=dec_bytes / (dec_ms * 1e-3) / 1e9 / pk["hbm_gbs"]),
                append=app)
    if big is not None:
        line["cfg4"] = big
        line["cfg3"] = sweep3
        line["cfg2"] = v2
    if not args.no_cpu_baseline:
        from oracle import gsrq_oracle as o
        t0 = time.perf_counter()
        oracle_step(x_np, w_np, c)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = dict(value=G * T / dt, unit=UNIT, cores=o.n_threads(), kind="oracle",
                                    sample=f"whole cfg{c.cfg} step once ({dt:.1f} s)")
    print(json.dumps(line))


if __name__ == "__main__":
    main()
