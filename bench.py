#!/usr/bin/env python
"""bench.py -- one JSON line per run (DESIGN.md section 9 says what each key means).

Headline workload = BASELINE.json config 4, the largest single-GPU configuration: one layer's K AND V cache,
batch 8 x 131072 tokens x 8 KV heads x 128, bf16, head-inner layout (2.147 GB each); d=16, K=256, S=2, 10 Lloyd
iterations; codebooks fitted on a seeded 65,536-token sample per head, then full-cache encode and full-cache decode.
A "step" is that whole hot path for both tensors:
    for X in (K, V): for s in 0..S-1: gsrq_fit_stage(X, stage s, fit sample) ; gsrq_encode(X, stages [0,S)) ; gsrq_decode(X)
value = KV vectors (token x head, 2 x 8 x 1,048,576 per step) through the whole step per second, summed over ranks
(replicas: every rank works on its own layer).  Inputs are resident in HBM and far larger than L2 (no flush needed).
e2e is the same through gsrq_pipeline_host_batch on pinned HOST buffers (H2D of the tensors, D2H of codes, codebooks and
the decoded tensors inside the timed region).  Rank 0 also times BASELINE configs 1-3 and the encode-on-append
latency as extras (>= 20 repetitions each, median and min), and the CPU oracle on a bounded sample.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-extras] [--no-cpu-baseline]
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
CFG4_T, CFG4_NFIT = 8 * 131072, 65536
ORACLE_FIT_HEADS, ORACLE_SLICE_TOKENS = 2, 16384


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return dict(hbm_gbs=d["hbm_gbs"], bf16_tflops=d["bf16_tflops"], bf16_tflops_sustained=d["bf16_tflops_sustained"],
                    source="MEASURED_PEAKS.json")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback (B200_PROFILING.md)")


def csrc_hash() -> str:
    """sha256 over the library's kernel sources (names and contents, sorted): ties a committed ncu capture to the code it measured."""
    import hashlib
    h = hashlib.sha256()
    for p in sorted((ROOT / "paper_2607_01065_b200" / "csrc").glob("*.cu*")):
        h.update(p.name.encode()); h.update(p.read_bytes())
    return h.hexdigest()


def workload_config():
    """The `config` object of the JSON line: identical for both arms."""
    c = inputs.CONFIGS[4]
    return dict(workload=f"cfg4:{c.name} (one layer's K and V cache, head-inner)", tensors="k,v", G=c.G, T=CFG4_T, hd=c.hd,
                d=c.d, K=c.K, S=c.S, iters=c.iters, n_fit_tokens=CFG4_NFIT,
                l2="inputs 17x larger than L2: no flush needed", parallelism="replicas")


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


# ------------------------------------------------------------------------------------------------ oracle (CPU) legs
def oracle_sample_seconds(kind: str) -> dict:
    """The CPU oracle, as it stands, on a BOUNDED sample of the cfg-4 step for one tensor kind, scaled to the whole step.
    Sample: a numpy draw of the same recipe with 65,536 tokens x 8 heads; the S=2, 10-iteration fit of ORACLE_FIT_HEADS
    heads on all 524,288 rows of each (= one head's fit sample), and encode + decode of all 8 heads over the first
    ORACLE_SLICE_TOKENS tokens with those codebooks.  Whole-step estimate: fit time x 8 / heads + encode/decode time x
    1,048,576 / slice tokens (the oracle's cost is linear in heads and in tokens)."""
    from oracle import gsrq_oracle as o
    c = inputs.CONFIGS[4]
    gen = inputs.k_like if kind == "k" else inputs.v_like
    x = gen(c.G, CFG4_NFIT, c.hd, inputs.seed_of(4, kind))
    w = inputs.token_weights(CFG4_NFIT, inputs.seed_of(4, "w"))
    t0 = time.perf_counter()
    fit = o.gsrq_fit_encode(x[:ORACLE_FIT_HEADS], w, c.d, c.K, c.S, c.iters, seed=0, encode=False)
    t_fit = time.perf_counter() - t0
    sh = np.concatenate([fit["shapes"]] * (c.G // ORACLE_FIT_HEADS))
    ga = np.concatenate([fit["gains"]] * (c.G // ORACLE_FIT_HEADS))
    t0 = time.perf_counter()
    codes, _, _, _ = o.encode(x[:, :ORACLE_SLICE_TOKENS], sh, ga, c.d)
    o.decode(codes, sh, ga, c.hd, bf16=True)
    t_ed = time.perf_counter() - t0
    full = t_fit * c.G / ORACLE_FIT_HEADS + t_ed * CFG4_T / ORACLE_SLICE_TOKENS
    return dict(fit_s=t_fit, encode_decode_s=t_ed, whole_step_s_estimate=full)


def oracle_value(steps: int = 1):
    """KV vectors/s of the oracle for the whole cfg-4 step (K and V), from the bounded samples; returns value, description."""
    from oracle import gsrq_oracle as o
    o.build()
    c = inputs.CONFIGS[4]
    tot, cpu = 0.0, 0.0
    for _ in range(steps):
        for kind in ("k", "v"):
            r = oracle_sample_seconds(kind)
            tot += r["whole_step_s_estimate"]
            cpu += r["fit_s"] + r["encode_decode_s"]
    val = steps * 2 * c.G * CFG4_T / tot
    desc = (f"per tensor (k, v): oracle fit of {ORACLE_FIT_HEADS} of 8 heads on 524,288 fit rows each + encode/decode of 8 heads x "
            f"{ORACLE_SLICE_TOKENS} tokens, scaled linearly to 8 heads / 1,048,576 tokens; {cpu / steps:.1f} s of CPU work per step")
    return val, tot / steps, desc, o.n_threads()


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, same config / metric (rank 0 only)."""
    for _ in range(min(args.warmup, 1)):
        oracle_sample_seconds("k")
    val, step_s, desc, cores = oracle_value(args.steps)
    line = dict(metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=step_s * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", impl="reference", config=workload_config(),
                cpu_baseline=dict(value=val, unit=UNIT, cores=cores, kind="oracle", sample=desc),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ replica helpers
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


def timed(f, reps=20, warm=3, flush=None):
    """CUDA-event timing of f on the current stream: `warm` untimed calls, `reps` timed ones; (median ms, min ms)."""
    for _ in range(warm):
        f()
    ts = []
    for _ in range(reps):
        if flush is not None:
            flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); f(); b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return float(np.median(ts)), float(np.min(ts))


# ------------------------------------------------------------------------------------------------ extras (rank 0)
def run_small_cfg(B, pk, cfg, kind, flush):
    """BASELINE configs 1 / 2 / 3 for one tensor kind (8 x T x 128 bf16, fit on all tokens, L2 flushed between repetitions):
    the whole step (per stage: fit + fused encode [0, s]; then decode), and encode / decode for every prefix S' = 1..S."""
    c = inputs.CONFIGS[cfg]
    G, T, hd, d, K, S, iters = c.G, c.T, c.hd, c.d, c.K, c.S, c.iters
    M = hd // d
    gen = inputs.k_like if kind == "k" else inputs.v_like
    x = torch.from_numpy(gen(G, T, hd, inputs.seed_of(cfg, kind))).to(torch.bfloat16).cuda()
    w = torch.from_numpy(inputs.token_weights(T, inputs.seed_of(cfg, "w"))).cuda()
    view = B.view_of(x, d)
    shapes = torch.zeros(G, S, K, d, device="cuda")
    gains = torch.zeros(G, S, K, device="cuda")
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, S, 0)
    codes = torch.zeros(S, G, T * M, dtype=torch.uint8, device="cuda")
    residual = torch.zeros(G, T * M, d, device="cuda")
    out = torch.empty_like(x)
    rows = G * T * M

    def fit_all():
        for s in range(S):
            B.gsrq_fit_stage(x, view, w, 0, None, cb, s, residual if s else None, iters, 0, ws, want_stats=False)
            B.gsrq_encode(x, view, cb, 0, s + 1, codes, residual if s + 1 < S else None, ws)

    def step():
        fit_all()
        B.gsrq_decode(codes, cb, S, out, view)

    step_ms, step_min = timed(step, flush=flush)
    fit_ms, fit_min = timed(fit_all, flush=flush)
    # weighted distortion after each stage, relative to the input's weighted energy (reading c-N)
    w_rows = w.repeat_interleave(M).double()
    e0 = float((w_rows[None] * (x.float().reshape(G, T * M, d).double() ** 2).sum(-1)).sum())
    dist = []
    for n in range(1, S + 1):
        B.gsrq_encode(x, view, cb, 0, n, codes, residual, ws)
        dist.append(float((w_rows[None] * (residual.double() ** 2).sum(-1)).sum()) / e0)
    sweep = []
    for n in range(1, S + 1):
        em, emin = timed(lambda: B.gsrq_encode(x, view, cb, 0, n, codes, None, ws), flush=flush)
        dm, dmin = timed(lambda: B.gsrq_decode(codes, cb, n, out, view), flush=flush)
        by = rows * n + rows * 2 * d
        sweep.append(dict(S=n, bits_per_element=n * 8.0 / d, encode_ms=em, encode_ms_min=emin,
                          encode_kv_vectors_per_s=G * T / (em * 1e-3),
                          encode_tensor_frac=2.0 * K * d * rows * n / (em * 1e-3) / 1e12 / pk["bf16_tflops_sustained"],
                          decode_ms=dm, decode_ms_min=dmin, decode_gb_per_s=by / (dm * 1e-3) / 1e9,
                          decode_frac_of_copy_bw=by / (dm * 1e-3) / 1e9 / pk["hbm_gbs"], rel_weighted_distortion=dist[n - 1]))
    floor_ms = (iters + 2) * S * max(2.0 * K * d * rows / (pk["bf16_tflops_sustained"] * 1e12), rows * 33.0 / (pk["hbm_gbs"] * 1e9)) * 1e3
    return dict(workload=f"cfg{cfg}:{kind}-cache-8x{T}x128, S={S}, {iters} iterations, fit on all tokens; L2 flushed per repetition"
                         f" ({x.numel() * 2 / 1e6:.0f} MB tensor: effective GB/s)",
                reps=20, step_ms=step_ms, step_ms_min=step_min, kv_vectors_per_s=G * T / (step_ms * 1e-3),
                fit_and_stage_encodes_ms=fit_ms, fit_and_stage_encodes_ms_min=fit_min,
                fit_floor_ms=floor_ms, sweep=sweep)


def run_append(B):
    """Encode-on-append (PAPER.md:443 (i)): latency of quantising the newest token(s) of a batch of sequences (cfg-1 layer)."""
    c = inputs.CONFIGS[1]
    G, T, hd, d, K, S = c.G, c.T, c.hd, c.d, c.K, c.S
    M = hd // d
    x = torch.from_numpy(inputs.k_like(G, T, hd, inputs.seed_of(1, "k"))).to(torch.bfloat16).cuda()
    gen = torch.Generator(device="cuda"); gen.manual_seed(5)
    sh = torch.nn.functional.normalize(torch.randn(G, S, K, d, device="cuda", generator=gen), dim=-1).contiguous()
    ga = torch.rand(G, S, K, device="cuda", generator=gen).contiguous()
    cb = B.codebook_of(sh, ga)
    codes = torch.zeros(S, G, T * M, dtype=torch.uint8, device="cuda")
    app = []
    for n_new in (8, 16, 32):
        chunk = x[:, :n_new]
        cv = B.view_of(chunk, d)

        def f():
            for _ in range(20):
                B.gsrq_encode_append(chunk, cv, cb, S, codes, T * M, 0)

        md, mn = timed(f, reps=20)
        app.append(dict(new_tokens=n_new, us_per_call=md * 1e3 / 20, us_per_call_min=mn * 1e3 / 20))
    return app


def run_d128(B, pk):
    """The paper's own operating point: D = 128, K = 256, R = 12 stages (0.75 bits per element) on a K-like
    8 x 32768 x 128 bf16 layer: 12 fits (10 iterations, each followed by the encode of that one stage, which feeds the next fit), the 12-stage
    encode, the decode, and the tcgen05 scoring pass alone (per-class CUDA-event time of one encode)."""
    G, T, hd, d, K, S, iters = 8, 32768, 128, 128, 256, 12, 10
    x = torch.from_numpy(inputs.k_like(G, T, hd, inputs.seed_of(3, "k"))).to(torch.bfloat16).cuda()
    w = torch.from_numpy(inputs.token_weights(T, inputs.seed_of(3, "w"))).cuda()
    view = B.view_of(x, d)
    sh = torch.zeros(G, S, K, d, device="cuda"); ga = torch.zeros(G, S, K, device="cuda")
    cb = B.codebook_of(sh, ga); ws = B.workspace(view, K, S, 0)
    codes = torch.zeros(S, G, T, dtype=torch.uint8, device="cuda")
    res = torch.zeros(G, T, d, device="cuda"); out = torch.empty_like(x)

    def fit_all():
        for s in range(S):
            B.gsrq_fit_stage(x, view, w, 0, None, cb, s, res if s else None, iters, 0, ws, want_stats=False)
            B.gsrq_encode(x, view, cb, s, s + 1, codes, res, ws)   # stage s only: the planes < s are read back to rebuild the residual, not re-encoded

    fit_ms, fit_min = timed(fit_all, reps=3, warm=1)
    enc_ms, enc_min = timed(lambda: B.gsrq_encode(x, view, cb, 0, S, codes, None, ws), reps=20)
    dec_ms, dec_min = timed(lambda: B.gsrq_decode(codes, cb, S, out, view), reps=20)
    B.gsrq_profile_enable(True)
    B.gsrq_encode(x, view, cb, 0, S, codes, None, ws)
    torch.cuda.synchronize()
    prof = B.gsrq_profile_read()
    B.gsrq_profile_enable(False)
    rows = G * T
    score_ms = prof["score"][0] / max(prof["score"][1], 1)
    flops = 2.0 * K * d * rows
    rel = float(((out.float() - x.float()) ** 2).sum() / (x.float() ** 2).sum())
    return dict(workload="d128: k-cache-8x32768x128, D=128, K=256, R=12 (0.75 bit/element), 10 iterations, fit on all tokens",
                fit_12_stages_with_stage_encodes_ms=fit_ms, fit_ms_min=fit_min, encode_12_stages_ms=enc_ms, encode_ms_min=enc_min,
                encode_kv_vectors_per_s=G * T / (enc_ms * 1e-3), encode_algorithmic_tflops=flops * S / (enc_ms * 1e-3) / 1e12,
                decode_ms=dec_ms, decode_ms_min=dec_min, decode_gb_per_s=rows * (S + 2 * d) / (dec_ms * 1e-3) / 1e9,
                scoring_pass=dict(kernel="tc::k_score_tc_wide<2> (tcgen05, SWIZZLE_128B operands)", ms_per_launch=score_ms,
                                  algorithmic_tflops=flops / (score_ms * 1e-3) / 1e12,
                                  frac_of_sustained_bf16_peak=flops / (score_ms * 1e-3) / 1e12 / pk["bf16_tflops_sustained"],
                                  note="17 (stage 0, bf16-exact rows) or 25 (residual stages) M128xN256xK16 MMAs per 128-row tile for 8 "
                                       "algorithmic ones: ncu tensor-pipe utilisation in profiles/r2_ncu_summaries.md"),
                encode_ms_by_class={k: v[0] for k, v in prof.items() if v[1]}, rel_residual_energy=rel)


def bf16_attention_baseline(Bq, ctx, G, Hq, hd, gen):
    """MEASURED library baselines for the same decoding step on an uncompressed bf16 KV cache (the paper's FP16 column):
    torch's scaled_dot_product_attention (the n_rep query heads of a KV head presented as n_rep query positions, so no head is
    replicated) and flash-attn's split-KV decode kernel when it runs on this GPU.  Library code, not this repo's: context only.
    The keys are taken as already rotated (a bf16 cache stores post-RoPE keys), so there is one number per (batch, context)."""
    out = {}
    n_rep = Hq // G
    k = torch.randn(Bq, G, ctx, hd, device="cuda", generator=gen).bfloat16()
    v = torch.randn(Bq, G, ctx, hd, device="cuda", generator=gen).bfloat16()
    q = torch.randn(Bq, G, n_rep, hd, device="cuda", generator=gen).bfloat16()
    try:
        f = lambda: torch.nn.functional.scaled_dot_product_attention(q, k, v)
        md, mn = timed(f, reps=20)
        out["torch_sdpa"] = dict(us=md * 1e3, us_min=mn * 1e3)
    except Exception as e:   # noqa: BLE001 -- a baseline that cannot run is reported, not fatal
        out["torch_sdpa"] = dict(error=str(e)[:200])
    try:
        from flash_attn import flash_attn_with_kvcache
        kc, vc = k.transpose(1, 2).contiguous(), v.transpose(1, 2).contiguous()   # [B][ctx][G][hd]
        q4 = q.reshape(Bq, 1, Hq, hd).contiguous()
        lens = torch.full((Bq,), ctx, dtype=torch.int32, device="cuda")
        f = lambda: flash_attn_with_kvcache(q4, kc, vc, cache_seqlens=lens)
        md, mn = timed(f, reps=20)
        out["flash_attn_with_kvcache"] = dict(us=md * 1e3, us_min=mn * 1e3)
        del kc, vc
    except Exception as e:   # noqa: BLE001
        out["flash_attn_with_kvcache"] = dict(error=str(e)[:200])
    del k, v, q
    torch.cuda.empty_cache()
    return out


def run_attention(B, pk):
    """Decode fused into attention (PAPER.md:443 (ii)): one decoding step of LLaMA-3-8B-shaped GQA (32 query / 8 KV heads, head_dim 128)
    straight from the GSRQ codes, for the batch / context pairs of the paper's latency tables: the d = 16, S = 2 codes
    of the headline config (table-lookup kernels) and the paper's own operating point D = 128, R = 12 (0.75 bits per element; the
    dequantising kernel).  Each leg sits beside MEASURED library attention on a bf16 cache of the same shape."""
    G, Hq, hd, K = 8, 32, 128, 256
    outl = []
    for Bq, ctx in ((8, 1024), (32, 1024), (1, 131072), (8, 131072)):
        T = Bq * ctx
        gen = torch.Generator(device="cuda"); gen.manual_seed(0)
        q = torch.randn(Bq, Hq, hd, device="cuda", generator=gen)
        start = (torch.arange(Bq, device="cuda") * ctx).to(torch.int64)
        length = torch.full((Bq,), ctx, dtype=torch.int64, device="cuda")
        o_ = torch.zeros(Bq, Hq, hd, device="cuda")
        base = bf16_attention_baseline(Bq, ctx, G, Hq, hd, gen)
        for d, S in ((16, 2), (128, 12)):
            M = hd // d
            kc = torch.randint(0, 256, (S, G, T * M), dtype=torch.uint8, device="cuda", generator=gen)
            vc = torch.randint(0, 256, (S, G, T * M), dtype=torch.uint8, device="cuda", generator=gen)
            sh = torch.nn.functional.normalize(torch.randn(G, S, K, d, device="cuda", generator=gen), dim=-1).contiguous()
            ga = torch.rand(G, S, K, device="cuda", generator=gen).contiguous()
            cb = B.codebook_of(sh, ga)
            for theta in (0.0, 500000.0):
                ws = B.gsrq_attention_decode(q, kc, cb, S, vc, cb, S, T * M, start, length, ctx, G, d, hd ** -0.5, theta, o_)
                md, mn = timed(lambda: B.gsrq_attention_decode(q, kc, cb, S, vc, cb, S, T * M, start, length, ctx, G, d, hd ** -0.5, theta, o_, ws),
                               reps=20 if d == 16 else 5)
                code_bytes = 2 * S * G * T * M
                outl.append(dict(batch=Bq, context=ctx, d=d, stages=S, rope=theta > 0, us=md * 1e3, us_min=mn * 1e3, code_bytes=code_bytes,
                                 codes_gb_per_s=code_bytes / (md * 1e-3) / 1e9, frac_of_copy_bw_on_code_bytes=code_bytes / (md * 1e-3) / 1e9 / pk["hbm_gbs"],
                                 bf16_cache_bytes=2 * G * T * hd * 2, us_to_read_bf16_cache_at_copy_bw=2 * G * T * hd * 2 / (pk["hbm_gbs"] * 1e9) * 1e6,
                                 bf16_attention_measured=base,
                                 speedup_over_measured_bf16_attention={k: v["us"] / (md * 1e3) for k, v in base.items() if "us" in v}))
            del kc, vc
        torch.cuda.empty_cache()
    return outl


def run_cluster(B):
    """GSKM against the K-means baseline on x ~ N(0, I_D), N = 10,000 (Fig. 4): two points of each sweep."""
    from paper_2607_01065_b200 import fig4_sweep
    t0 = time.perf_counter()
    rows = fig4_sweep.sweep(settings=[(128, 2048), (256, 2048), (256, 256)], iters=25)
    return dict(seconds=time.perf_counter() - t0, rows=rows)


# ------------------------------------------------------------------------------------------------ main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the config 1-3 / append legs (rank 0)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg (profiling aid)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        if rank == 0:
            run_reference(args)
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
    pk = peaks()
    c = inputs.CONFIGS[4]
    G, hd, d, K, S, iters = c.G, c.hd, c.d, c.K, c.S, c.iters
    T, n_fit, M = CFG4_T, CFG4_NFIT, c.hd // c.d
    rows = G * T * M
    rows_fit = G * n_fit * M

    # ---- inputs: one layer's K and V cache, drawn on the device (replicas: rank r draws its own layer) ----
    tens = {}
    for kind in ("k", "v"):
        dd = inputs.cfg4_device(kind, T, n_fit, seed=rank_seed(4, kind, rank))
        tens[kind] = dd
    view = B.view_of(tens["k"]["x"], d, head_inner=True)
    cbs = {}
    for kind in ("k", "v"):
        sh = torch.zeros(G, S, K, d, device="cuda")
        ga = torch.zeros(G, S, K, device="cuda")
        cbs[kind] = (B.codebook_of(sh, ga), sh, ga)
    ws = B.workspace(view, K, S, n_fit)
    codes = {kind: torch.zeros(S, G, T * M, dtype=torch.uint8, device="cuda") for kind in ("k", "v")}
    out = torch.empty_like(tens["k"]["x"])

    def fit(kind):
        t = tens[kind]
        for s in range(S):   # the stage-1 fit re-derives its residual on the fit rows from kv + the stage-0 codebook
            B.gsrq_fit_stage(t["x"], view, t["w"], 0, t["fit_tokens"], cbs[kind][0], s, None, iters, 0, ws, want_stats=False)

    def encode(kind):
        B.gsrq_encode(tens[kind]["x"], view, cbs[kind][0], 0, S, codes[kind], None, ws)

    def decode(kind):
        B.gsrq_decode(codes[kind], cbs[kind][0], S, out, view)

    def step():
        for kind in ("k", "v"):
            fit(kind); encode(kind); decode(kind)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()                          # nvidia-smi takes a moment to come up: start it before the warm-up
    warm = max(args.warmup, 3)
    for _ in range(warm):
        step()
    barrier()
    t_region0 = time.perf_counter()
    l0 = B.gsrq_launch_count()
    evs = []
    for _ in range(args.steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); step(); b.record()
        evs.append((a, b))
    barrier()
    t_region1 = time.perf_counter()
    launches = B.gsrq_launch_count() - l0
    ms = sum(a.elapsed_time(b) for a, b in evs)
    units = 2 * G * T
    value, max_s = whole_job_value(ms * 1e-3 / args.steps, units, world, "cuda")
    ms_per_step = max_s * 1e3
    clocks = sampler.finish(t_region0, t_region1)

    # ---- per-kernel device time of one step, measured live with CUDA events around every launch ----
    B.gsrq_profile_enable(True)
    step()
    torch.cuda.synchronize()
    prof = B.gsrq_profile_read()
    B.gsrq_profile_enable(False)
    # the three parts for both tensors: >= 20 repetitions, median and min
    parts = {}
    for kind in ("k", "v"):
        f_md, f_mn = timed(lambda: fit(kind), reps=20, warm=1)
        e_md, e_mn = timed(lambda: encode(kind), reps=20, warm=1)
        d_md, d_mn = timed(lambda: decode(kind), reps=20, warm=1)
        parts[kind] = dict(fit_ms=f_md, fit_ms_min=f_mn, encode_ms=e_md, encode_ms_min=e_mn, decode_ms=d_md, decode_ms_min=d_mn)
    # sanity: decode(encode(x)) must be closer to x than 0 is (relative residual energy < 1), V tensor, first 4096 tokens
    xv = tens["v"]["x"][:4096].float()
    rel_err = float(((out[:4096].float() - xv) ** 2).sum() / (xv ** 2).sum())

    # ---- end to end through the host-buffer C-ABI call: H2D + fit + encode + decode + D2H ----
    e2e = None
    if not args.no_e2e:
        host = {kind: dict(x=tens[kind]["x"].cpu().pin_memory(), w=tens[kind]["w"].cpu().pin_memory(),
                           fit=tens[kind]["fit_tokens"].cpu().pin_memory()) for kind in ("k", "v")}
        kinds = ("k", "v")
        sh_h = [torch.empty(G, S, K, d).pin_memory() for _ in kinds]; ga_h = [torch.empty(G, S, K).pin_memory() for _ in kinds]
        co_h = [torch.empty(S, G, T * M, dtype=torch.uint8).pin_memory() for _ in kinds]
        out_h = [torch.empty(T, G, hd, dtype=torch.bfloat16).pin_memory() for _ in kinds]
        del out, codes
        torch.cuda.empty_cache()

        def e2e_step():   # one call for the layer's K and V cache: V uploads while K is fitted, encoded, decoded and downloaded
            B.gsrq_pipeline_host_batch([host[k_]["x"] for k_ in kinds], view, [host[k_]["w"] for k_ in kinds], [host[k_]["fit"] for k_ in kinds],
                                       K, S, iters, 0, sh_h, ga_h, co_h, out_h)

        e2e_step()
        barrier()
        n_e2e = max(3, args.steps // 3)
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            e2e_step()
        barrier()
        e2e_s = (time.perf_counter() - t0) / n_e2e
        e2e_val, _ = whole_job_value(e2e_s, units, world, "cuda")
        h2d = sum(h["x"].numel() * 2 + h["w"].numel() * 4 + h["fit"].numel() * 8 for h in host.values())
        d2h = sum(sh_h[i].numel() * 4 + ga_h[i].numel() * 4 + co_h[i].numel() + out_h[i].numel() * 2 for i in range(len(kinds)))
        e2e = dict(value=e2e_val, unit=UNIT, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h, ms_per_step=e2e_s * 1e3,
                   steps=n_e2e, call="gsrq_pipeline_host_batch (K and V in one call, pinned host buffers, fit_tokens given)")
        B.gsrq_release_host_pool()
        del host, sh_h, ga_h, co_h, out_h
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()      # no collective below: the remaining legs run on rank 0 alone
    if rank != 0:
        return

    # ---- rooflines: algorithmic work per launch / live launch duration ----
    tot_ms = sum(v[0] for v in prof.values())

    traffic_file = "profiles/r3_traffic.csv"
    traffic_stale = [None]

    def ncu_traffic(cls):
        """dram__bytes_read.sum + dram__bytes_write.sum per launch of the class (average over its launches per tensor), from the committed
        ncu --set full capture of this command (not measured in this run).  The capture names the kernel sources it was taken on
        (column csrc_sha256 = csrc_hash()); when they have changed since, the figure is stale and None is reported instead."""
        try:
            import csv
            with open(ROOT / traffic_file) as f:
                rws = [r for r in csv.DictReader(f) if r["class"] == cls]
            if not rws or any(r.get("csrc_sha256") != csrc_hash() for r in rws):
                traffic_stale[0] = True
                return None
            n_l = sum(int(r["launches_per_tensor"]) for r in rws)
            return sum((int(r["dram_bytes_read"]) + int(r["dram_bytes_write"])) * int(r["launches_per_tensor"]) for r in rws) / n_l if n_l else None
        except (OSError, KeyError, ValueError):
            return None

    def kern(name, cls, bound, work_per_launch, unit, note):
        ms_c, n = prof[cls]
        per = ms_c / max(n, 1)
        peak = pk["bf16_tflops_sustained"] if bound == "tensor" else pk["hbm_gbs"]
        ach = work_per_launch / (per * 1e-3) / (1e12 if bound == "tensor" else 1e9) if per > 0 else 0.0
        return dict(bound=bound, kernel=name, achieved=ach, peak=peak, unit=unit, frac=ach / peak, traffic=ncu_traffic(cls),
                    traffic_note=f"bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum, class average) from the committed ncu --set full capture "
                                 f"of this command ({traffic_file}); not measured in this run; null when there is no capture of the current kernel "
                                 f"sources (csrc hash {csrc_hash()[:12]})",
                    algorithmic_per_launch=work_per_launch, ms_per_launch=per, launches=n,
                    share_of_step=ms_c / tot_ms if tot_ms else None, note=note)

    kerns = [
        kern("tc::k_fit_tc (persistent fit: tcgen05 scoring + arg-max, fp64 reduction, merge, Eq. 7/8; all passes of a stage)", "score",
             "tensor", 2.0 * K * d * rows_fit * (iters + 1), "TFLOP/s",
             "8192 flops per sub-vector per pass x 4,194,304 fit rows x 11 passes per launch (one launch per stage and tensor)"),
        kern("tc::k_encode_tc (fused S-stage encode; also the stage-1 residual derivation on the fit rows)", "encode", "tensor",
             2.0 * K * d * (rows * S + rows_fit * 1) / 2.0, "TFLOP/s",
             "class average over its two launches per tensor: full-cache S=2 encode (67,108,864 rows) and the 1-stage derivation on the fit rows"),
        kern("k_decode_fast (gather + sum of S scaled codewords)", "decode", "hbm", float(rows * (S + 2 * d)), "GB/s",
             "S + 32 bytes per sub-vector x 67,108,864 rows"),
    ]
    dom = max(kerns, key=lambda kk: kk["share_of_step"] or 0.0)
    roofline = dict(dom)
    roofline["peak_source"] = pk["source"] + (" (sustained bf16: kernel timed inside a long step)" if dom["bound"] == "tensor"
                                              else " (copy bandwidth)")
    roofline["by_class_ms_per_step"] = {k: dict(ms=v[0], launches=v[1]) for k, v in prof.items()}
    roofline["other_kernels"] = [kk for kk in kerns if kk is not dom]
    # whole parts against their floors (per tensor)
    fit_floor_ms = (iters + 2) * S * max(2.0 * K * d * rows_fit / (pk["bf16_tflops_sustained"] * 1e12),
                                         rows_fit * 33.0 / (pk["hbm_gbs"] * 1e9)) * 1e3
    enc_floor_ms = max(2.0 * K * d * rows * S / (pk["bf16_tflops_sustained"] * 1e12), rows * (2 * d + S) / (pk["hbm_gbs"] * 1e9)) * 1e3
    dec_bytes = rows * (S + 2 * d)
    for kind in ("k", "v"):
        pp = parts[kind]
        pp["fit_floor_ms"] = fit_floor_ms
        pp["fit_frac_of_floor"] = fit_floor_ms / pp["fit_ms"]
        pp["encode_floor_ms"] = enc_floor_ms
        pp["encode_kv_vectors_per_s"] = G * T / (pp["encode_ms"] * 1e-3)
        pp["encode_tensor_frac"] = 2.0 * K * d * rows * S / (pp["encode_ms"] * 1e-3) / 1e12 / pk["bf16_tflops_sustained"]
        pp["decode_gb_per_s"] = dec_bytes / (pp["decode_ms"] * 1e-3) / 1e9
        pp["decode_frac_of_copy_bw"] = pp["decode_gb_per_s"] / pk["hbm_gbs"]
        pp["decode_frac_of_nominal_hbm_7700"] = pp["decode_gb_per_s"] / 7700.0
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=warm,
                ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="bf16 in, fp32/fp64 arithmetic", data="synthetic", impl="ours", config=workload_config(),
                clocks=clocks, gpu_launches=int(launches), e2e=e2e, roofline=roofline, parts=parts,
                rel_residual_energy_v_first_4096_tokens=rel_err)
    if not args.no_extras:
        del tens, ws
        torch.cuda.empty_cache()
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
        extras = {}
        for cfg, kinds in ((1, ("k",)), (2, ("v",)), (3, ("k", "v"))):
            for kind in kinds:
                extras[f"cfg{cfg}_{kind}"] = run_small_cfg(B, pk, cfg, kind, flush)
                torch.cuda.empty_cache()
        extras["append"] = run_append(B)
        extras["d128"] = run_d128(B, pk)
        torch.cuda.empty_cache()
        extras["attention_decode"] = run_attention(B, pk)
        extras["fig4_sweep_excerpt"] = run_cluster(B)
        line["extras"] = extras
    if not args.no_cpu_baseline:
        val, step_s, desc, cores = oracle_value(1)
        line["cpu_baseline"] = dict(value=val, unit=UNIT, cores=cores, kind="oracle", sample=desc,
                                    whole_step_s_estimate=step_s)
    print(json.dumps(line))


if __name__ == "__main__":
    main()
