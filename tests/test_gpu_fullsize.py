"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times, and the edge
cases of the tensor-core encode and the bandwidth decode.  Run with `-m gpu` on a B200.

cfg 1 and cfg 2 are small enough for the oracle to run whole (seconds on the box's cores), so they are
compared element by element.  cfg 4's layout is checked at 65,536 tokens x 8 heads (134 MB) on sampled
tokens: a token's codes depend on that token's rows only, so the oracle encodes the sample alone."""
import numpy as np
import pytest
import torch

from paper_2607_01065_b200.pipeline import gpu_decode, gpu_gsrq, stats_np, to_device
from oracle import gsrq_oracle as o
from paper_2607_01065_b200 import inputs
from test_gpu_parity import _check_free_running

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import __graft_entry__ as ge
    ge.build()
    from paper_2607_01065_b200 import binding
    return binding


def test_cfg1_full_size_bench_flow():
    """BASELINE config 1 whole (8 x 4096 x 128, K=256, S=2, 20 iterations), bench.py's call sequence."""
    dd = inputs.make(1)
    c = dd["config"]
    got, ref = _check_free_running(dd, c.K, c.S, c.iters, "bf16", prefix_encode=True)
    assert np.array_equal(got["codes"], ref["codes"])           # identical trajectories, not merely within tolerance
    assert np.array_equal(got["shapes"], ref["shapes"]) and np.array_equal(got["gains"], ref["gains"])
    dec = gpu_decode(got["codes_dev"], got["cb"], c.S, c.G, c.T, c.hd, c.d, dtype="bf16")
    want, _ = o.decode(got["codes"], got["shapes"], got["gains"], c.hd, bf16=True)
    assert np.array_equal(dec, want)


def test_cfg2_full_size():
    """BASELINE config 2 whole (V-like 8 x 16384 x 128, S=1, 20 iterations) + decode of the layer."""
    dd = inputs.make(2)
    c = dd["config"]
    got, ref = _check_free_running(dd, c.K, c.S, c.iters, "bf16", prefix_encode=True)
    dec = gpu_decode(got["codes_dev"], got["cb"], c.S, c.G, c.T, c.hd, c.d, dtype="bf16")
    want, _ = o.decode(got["codes"], got["shapes"], got["gains"], c.hd, bf16=True)
    assert np.array_equal(dec, want)


def test_cfg4_layout_sampled_encode_decode(B):
    """Head-inner [T][G][hd] tensor of 65,536 tokens: codebooks fitted on a 4,096-token sample per head
    (both sides), full encode + decode on the GPU, oracle on 3,000 sampled tokens."""
    T, n_fit, S, K, iters = 65536, 4096, 2, 256, 4
    c = inputs.CONFIGS[4]
    x = inputs.k_like(c.G, T, c.hd, inputs.seed_of(4, "k"))
    w = inputs.token_weights(T, inputs.seed_of(4, "w"))
    fit = inputs.fit_sample(c.G, T, n_fit, inputs.seed_of(4, "fit"))
    got = gpu_gsrq(x, w, c.d, K, S, iters, dtype="bf16", fit_tokens=fit, head_inner=True, pass_residual=False,
                   want_residual=False)
    ref = o.gsrq_fit_encode(x, w, c.d, K, S, iters, seed=0, fit_tokens=fit, encode=False)
    rng = np.random.default_rng(7)
    tok = np.sort(rng.choice(T, 3000, replace=False))
    assert np.abs(got["shapes"] - ref["shapes"]).max() <= 1e-4 and np.abs(got["gains"] - ref["gains"]).max() <= 1e-4
    assert np.array_equal(got["shapes"], ref["shapes"]) and np.array_equal(got["gains"], ref["gains"])
    # oracle encode of the sampled tokens with the GPU's codebooks (fixed-codebook encode is per row)
    codes_o, _, best, second = o.encode(x[:, tok], got["shapes"], got["gains"], c.d)
    M = c.hd // c.d
    rows = (tok[:, None] * M + np.arange(M)[None]).reshape(-1)
    codes_g = got["codes"][:, :, rows]
    assert np.array_equal(codes_g, codes_o)
    dec = gpu_decode(got["codes_dev"], got["cb"], S, c.G, T, c.hd, c.d, dtype="bf16", head_inner=True)
    want, _ = o.decode(codes_o, got["shapes"], got["gains"], c.hd, bf16=True)
    assert np.array_equal(dec[:, tok], want)


@pytest.mark.parametrize("hd,T,K,S", [(64, 150, 256, 2), (32, 333, 37, 4), (256, 40, 256, 3), (16, 1000, 256, 1)])
def test_tc_encode_shapes(B, hd, T, K, S):
    """Fused tensor-core encode for M = hd/16 in {1, 2, 4, 16}, ragged tile tails, K < 256, S up to 4."""
    rng = np.random.default_rng(hd + T)
    G = 3
    x = inputs.bf16_round(rng.standard_normal((G, T, hd)) * np.exp(0.5 * rng.standard_normal((G, T, 1))))
    sh = rng.standard_normal((G, S, K, 16))
    sh = (sh / np.linalg.norm(sh, axis=-1, keepdims=True)).astype(np.float32)
    ga = np.abs(rng.standard_normal((G, S, K)) * (2.0 / (1 + np.arange(S))[None, :, None])).astype(np.float32)
    codes_o, res_o, _, _ = o.encode(x, sh, ga, 16)
    xd = to_device(x, "bf16")
    view = B.view_of(xd, 16)
    sh_d, ga_d = torch.from_numpy(sh).cuda(), torch.from_numpy(ga).cuda()   # keep alive: cb holds raw pointers
    cb = B.codebook_of(sh_d, ga_d)
    ws = B.workspace(view, K, S, -1)
    M = hd // 16
    codes = torch.zeros(S, G, T * M, dtype=torch.uint8, device="cuda")
    res = torch.zeros(G, T * M, 16, device="cuda")
    B.gsrq_encode(xd, view, cb, 0, S, codes, res, ws)
    torch.cuda.synchronize()
    assert np.array_equal(codes.cpu().numpy(), codes_o)
    assert np.array_equal(res.cpu().numpy(), res_o)


def test_tc_encode_all_rows_ambiguous(B):
    """Duplicate codewords make every row an exact tie: all rows go through the exact path, lowest index wins."""
    rng = np.random.default_rng(3)
    G, T, hd, K, S = 2, 200, 128, 64, 2
    x = inputs.bf16_round(rng.standard_normal((G, T, hd)))
    sh = rng.standard_normal((G, S, K // 2, 16))
    sh = (sh / np.linalg.norm(sh, axis=-1, keepdims=True)).astype(np.float32)
    sh = np.concatenate([sh, sh], axis=2)                      # codeword k + K/2 == codeword k
    ga = np.abs(rng.standard_normal((G, S, K // 2))).astype(np.float32)
    ga = np.concatenate([ga, ga], axis=2)
    codes_o, res_o, _, _ = o.encode(x, sh, ga, 16)
    assert codes_o.max() < K // 2
    xd = to_device(x, "bf16")
    view = B.view_of(xd, 16)
    sh_d, ga_d = torch.from_numpy(sh).cuda(), torch.from_numpy(ga).cuda()   # keep alive: cb holds raw pointers
    cb = B.codebook_of(sh_d, ga_d)
    ws = B.workspace(view, K, S, -1)
    codes = torch.zeros(S, G, T * 8, dtype=torch.uint8, device="cuda")
    res = torch.zeros(G, T * 8, 16, device="cuda")
    B.gsrq_encode(xd, view, cb, 0, S, codes, res, ws)
    torch.cuda.synchronize()
    assert np.array_equal(codes.cpu().numpy(), codes_o) and np.array_equal(res.cpu().numpy(), res_o)


@pytest.mark.parametrize("T,S,dtype,head_inner", [(100, 1, "bf16", False), (100, 2, "f32", False), (515, 3, "bf16", True),
                                                  (32, 4, "bf16", False), (31, 2, "bf16", False), (4096, 4, "bf16", True),
                                                  (300, 7, "bf16", True), (130, 12, "f32", False), (64, 14, "bf16", False)])
def test_decode_bandwidth_path_and_tail(B, T, S, dtype, head_inner):
    """Decode: full 256-row chunks through k_decode_fast (1-4 stages: duplicated tables; 5-12: single-copy tables; more:
    generic kernel), the ragged tail through the generic kernel;
    N % 16 != 0 (T = 31... with M = 8 always a multiple of 8 only) falls back entirely.  Bit-exact."""
    rng = np.random.default_rng(T * 10 + S)
    G, hd, K = 2, 128, 256
    M = hd // 16
    sh = rng.standard_normal((G, S, K, 16))
    sh = (sh / np.linalg.norm(sh, axis=-1, keepdims=True)).astype(np.float32)
    ga = np.abs(rng.standard_normal((G, S, K))).astype(np.float32)
    codes = rng.integers(0, K, size=(S, G, T * M), dtype=np.uint8)
    sh_d, ga_d = torch.from_numpy(sh).cuda(), torch.from_numpy(ga).cuda()   # keep alive: cb holds raw pointers
    cb = B.codebook_of(sh_d, ga_d)
    cd = torch.from_numpy(codes).cuda()
    for n in range(1, S + 1):
        dec = gpu_decode(cd, cb, n, G, T, hd, 16, dtype=dtype, head_inner=head_inner)
        want, _ = o.decode(codes, sh, ga, hd, S_used=n, bf16=(dtype == "bf16"))
        assert np.array_equal(dec, want), (T, n)


def test_decision_margin_stress(B):
    """The filter's decision margin caps the competitor's gain by what can still beat the winner; stress it with
    gains spread over orders of magnitude (zeros included), rows from tiny to huge norms, zero rows and
    near-duplicate codewords, in both the 1-plane (bf16 rows) and 2-plane (fp32 residual) paths.  The result
    must equal the exact arg-max everywhere (ties -> lowest index)."""
    rng = np.random.default_rng(11)
    G, T, hd, K, S = 4, 2048, 128, 256, 2
    x = rng.standard_normal((G, T, hd)) * np.exp(1.5 * rng.standard_normal((G, T, 1)))
    x[:, ::97] = 0.0
    x[:, 5::211] *= 1e-3
    x = inputs.bf16_round(x)
    sh = rng.standard_normal((G, S, K, 16))
    sh[:, :, 128:192] = sh[:, :, 0:64] + 1e-4 * rng.standard_normal((G, S, 64, 16))   # near-duplicates
    sh = (sh / np.linalg.norm(sh, axis=-1, keepdims=True)).astype(np.float32)
    ga = np.exp(2.0 * rng.standard_normal((G, S, K))).astype(np.float32)
    ga[:, :, 128:192] = ga[:, :, 0:64]
    ga[:, :, 7::31] = 0.0
    codes_o, res_o, _, _ = o.encode(x, sh, ga, 16)
    xd = to_device(x, "bf16")
    view = B.view_of(xd, 16)
    sh_d, ga_d = torch.from_numpy(sh).cuda(), torch.from_numpy(ga).cuda()
    cb = B.codebook_of(sh_d, ga_d)
    ws = B.workspace(view, K, S, 0)
    codes = torch.zeros(S, G, T * 8, dtype=torch.uint8, device="cuda")
    res = torch.zeros(G, T * 8, 16, device="cuda")
    B.gsrq_encode(xd, view, cb, 0, S, codes, res, ws)          # fused tensor-core encode
    torch.cuda.synchronize()
    assert np.array_equal(codes.cpu().numpy(), codes_o) and np.array_equal(res.cpu().numpy(), res_o)
    # fit-path scoring kernel: stage 0 from the bf16 rows (1 plane), stage 1 from the fp32 residual (2 planes)
    idx = torch.zeros(G, T * 8, dtype=torch.uint8, device="cuda")
    B.gsrq_assign(xd, view, None, cb, 0, 0, idx, ws)
    assert np.array_equal(idx.cpu().numpy(), codes_o[0])
    _, res0, _, _ = o.encode(x, sh, ga, 16, stage_end=1)
    res0_d = torch.from_numpy(np.ascontiguousarray(res0)).cuda()
    B.gsrq_assign(xd, view, res0_d, cb, 1, 0, idx, ws)
    assert np.array_equal(idx.cpu().numpy(), codes_o[1])
    # projection mode (Alg. 1 l.2 assignment)
    B.gsrq_assign(xd, view, None, cb, 0, 1, idx, ws)
    rows = o.rows_of(x, 16)
    for g_ in range(G):
        a, _, _ = o.assign(rows[g_], sh[g_, 0], None)
        assert np.array_equal(idx[g_].cpu().numpy(), a.astype(np.uint8))


@pytest.mark.parametrize("dtype,hd,d,head_inner", [("bf16", 128, 16, True), ("bf16", 128, 16, False), ("f32", 64, 8, False), ("bf16", 64, 32, False)])
def test_encode_on_append_equals_batch_encode(B, dtype, hd, d, head_inner):
    """PAPER.md:443 (i): new tokens are quantised as they are generated.  Appending tokens 1, 3, 8, 32 at a time
    must fill the code planes exactly as one batch encode (and as the oracle) does."""
    rng = np.random.default_rng(5)
    G, T, K, S = 4, 140, 200, 3
    x = rng.standard_normal((G, T, hd)).astype(np.float32) * np.exp(0.4 * rng.standard_normal((G, T, 1))).astype(np.float32)
    if dtype == "bf16":
        x = inputs.bf16_round(x)
    sh = rng.standard_normal((G, S, K, d))
    sh = (sh / np.linalg.norm(sh, axis=-1, keepdims=True)).astype(np.float32)
    ga = np.abs(rng.standard_normal((G, S, K)) / (1 + np.arange(S))[None, :, None]).astype(np.float32)
    codes_o, _, _, _ = o.encode(x, sh, ga, d)
    M = hd // d
    xd = to_device(x, dtype, head_inner)
    sh_d, ga_d = torch.from_numpy(sh).cuda(), torch.from_numpy(ga).cuda()
    cb = B.codebook_of(sh_d, ga_d)
    codes = torch.full((S, G, T * M), 255, dtype=torch.uint8, device="cuda")
    t0 = 0
    for n_new in [1, 3, 8, 32, 1, 64, 31]:
        n_new = min(n_new, T - t0)
        chunk = xd[t0:t0 + n_new] if head_inner else xd[:, t0:t0 + n_new]
        B.gsrq_encode_append(chunk, B.view_of(chunk, d, head_inner), cb, S, codes, T * M, t0)
        t0 += n_new
    assert t0 == T
    torch.cuda.synchronize()
    assert np.array_equal(codes.cpu().numpy(), codes_o)
    with pytest.raises(B.GsrqError):
        B.gsrq_encode_append(chunk, B.view_of(chunk, d, head_inner), cb, S, codes, T * M, T)   # does not fit


@pytest.mark.parametrize("S,dtype,hd,K", [(8, "bf16", 128, 256), (10, "bf16", 64, 100), (5, "f32", 128, 256), (2, "f32", 16, 64)])
def test_tc_encode_chained_passes_and_fp32_rows(B, S, dtype, hd, K):
    """More than 4 stages run as chained tensor-core passes through an fp32 residual (the paper's deep residual
    quantisers: R = 12..32), and a dense fp32 tensor with d = 16 starts from fp32 rows: codes,
    residual and decode must equal the oracle, with and without a residual output."""
    rng = np.random.default_rng(S * 7 + hd)
    G, T = 3, 210
    x = rng.standard_normal((G, T, hd)) * np.exp(0.5 * rng.standard_normal((G, T, 1)))
    x = inputs.bf16_round(x) if dtype == "bf16" else x.astype(np.float32)
    sh = rng.standard_normal((G, S, K, 16))
    sh = (sh / np.linalg.norm(sh, axis=-1, keepdims=True)).astype(np.float32)
    ga = np.abs(rng.standard_normal((G, S, K)) * (2.0 / (1 + np.arange(S))[None, :, None])).astype(np.float32)
    codes_o, res_o, _, _ = o.encode(x, sh, ga, 16)
    xd = to_device(x, dtype)
    view = B.view_of(xd, 16)
    sh_d, ga_d = torch.from_numpy(sh).cuda(), torch.from_numpy(ga).cuda()
    cb = B.codebook_of(sh_d, ga_d)
    ws = B.workspace(view, K, S, -1)
    M = hd // 16
    for want_res in (True, False):
        codes = torch.zeros(S, G, T * M, dtype=torch.uint8, device="cuda")
        res = torch.zeros(G, T * M, 16, device="cuda") if want_res else None
        B.gsrq_encode(xd, view, cb, 0, S, codes, res, ws)
        torch.cuda.synchronize()
        assert np.array_equal(codes.cpu().numpy(), codes_o), (S, want_res)
        if want_res:
            assert np.array_equal(res.cpu().numpy(), res_o)
    dec = gpu_decode(codes, cb, S, G, T, hd, 16, dtype=dtype)
    want, _ = o.decode(codes_o, sh, ga, hd, bf16=(dtype == "bf16"))
    assert np.array_equal(dec, want)


def _sampled_encode_decode_check(B, x_dev, view, head_inner, cb, shapes, gains, S, tok, d=16):
    """Full-tensor encode + decode on the GPU; the oracle encodes / decodes the sampled tokens one by one with the same
    (GPU-fitted) codebooks.  A token's codes depend on that token's rows only."""
    G, T, hd = view.G, view.T, view.hd
    M = hd // d
    ws = B.workspace(view, cb.K, S, -1)
    codes = torch.zeros(S, G, T * M, dtype=torch.uint8, device="cuda")
    B.gsrq_encode(x_dev, view, cb, 0, S, codes, None, ws)
    out = torch.empty_like(x_dev)
    B.gsrq_decode(codes, cb, S, out, view)
    torch.cuda.synchronize()
    tok_d = torch.from_numpy(tok).cuda()
    xs = (x_dev[tok_d].permute(1, 0, 2) if head_inner else x_dev[:, tok_d]).float().cpu().numpy()      # [G][n][hd]
    outs = (out[tok_d].permute(1, 0, 2) if head_inner else out[:, tok_d]).float().cpu().numpy()
    rows = (tok_d[:, None] * M + torch.arange(M, device="cuda")[None]).reshape(-1)
    codes_s = codes[:, :, rows].cpu().numpy()
    codes_o, res_o, _, _ = o.encode(xs, shapes, gains, d, stage_end=S)
    assert np.array_equal(codes_s, codes_o)
    want, _ = o.decode(codes_o, shapes, gains, hd, S_used=S, bf16=True)
    assert np.array_equal(outs, want)
    assert int(codes.max()) < cb.K
    # x = (fp32) decode + residual on the sample, up to the fp32 rounding of the stage sums
    want32, _ = o.decode(codes_o, shapes, gains, hd, S_used=S, bf16=False)
    np.testing.assert_allclose(o.rows_of(want32, d) + res_o, o.rows_of(xs, d), atol=1e-4, rtol=1e-5)


def _oracle_fit_rows(rows, w_rows, K, S, iters, G):
    """The oracle's S-stage fit on compact fit rows [G][Nf][d] (a stage's residual on the fit rows depends on those rows
    only): Alg. 1 per group and stage, then the stage's encode to get the next residual.  Returns shapes, gains, stats."""
    d = rows.shape[-1]
    shapes = np.zeros((G, S, K, d), np.float32)
    gains = np.zeros((G, S, K), np.float32)
    stats = [[None] * S for _ in range(G)]
    for g_ in range(G):
        r = np.ascontiguousarray(rows[g_], dtype=np.float32)
        for st in range(S):
            f = o.fit_stage(r, w_rows[g_], K, iters, 0, group=g_, G=G, stage=st)
            shapes[g_, st], gains[g_, st], stats[g_][st] = f["shapes"], f["gains"], f
            if st + 1 < S:
                _, r, _, _ = o.encode_stage(r, f["shapes"], f["gains"])
    return shapes, gains, stats


def _assert_fit_matches(got_shapes, got_gains, got_stats, ref_shapes, ref_gains, ref_stats, G, S):
    """BASELINE criteria (b) codewords / gains within 1e-4 and (c) weighted distortion within 1e-4 relative -- here for every
    iteration's J, plus the discrete trajectory: iterations run, rows changed per iteration, empty clusters."""
    assert np.abs(got_shapes - ref_shapes).max() <= 1e-4
    assert np.abs(got_gains - ref_gains).max() <= 1e-4
    for st in range(S):
        for g_ in range(G):
            s_ref, s_got = ref_stats[g_][st], stats_np(got_stats[st], g_)
            assert s_got["iters_run"] == s_ref["iters_run"], (st, g_)
            np.testing.assert_allclose(s_got["J"], s_ref["J_assign"], rtol=1e-4)
            assert np.array_equal(s_got["changed"], s_ref["changed"]), (st, g_)
            assert s_got["n_empty_last"] == s_ref["n_empty_last"]


@pytest.mark.parametrize("kind", ["k", "v"])
def test_cfg4_full_size_fit_vs_oracle_then_sampled_encode_decode(B, kind):
    """BASELINE config 4 at its full size, as bench.py runs it: 8 x 131072 tokens x 8 heads x 128 bf16 (2.1 GB, head-inner),
    K-like and V-like.  The S = 2, 10-iteration fit on the 65,536-token sample per head (524,288 fit rows per head) is
    compared with the oracle run on the same bits (fit rows copied to the host): codebooks, per-iteration distortion,
    iterations and changed counts.  Then the full-cache encode and decode, checked on 2,048 sampled tokens against the
    oracle encoding them with the ORACLE's codebooks."""
    c = inputs.CONFIGS[4]
    G, hd, d, K, S, iters = c.G, c.hd, c.d, c.K, c.S, c.iters
    T, n_fit, M = 8 * 131072, 65536, c.hd // c.d
    dd = inputs.cfg4_device(kind, T, n_fit)
    x, w, fit = dd["x"], dd["w"], dd["fit_tokens"]
    view = B.view_of(x, d, head_inner=True)
    shapes = torch.zeros(G, S, K, d, device="cuda")
    gains = torch.zeros(G, S, K, device="cuda")
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, S, n_fit)
    stats = [B.gsrq_fit_stage(x, view, w, 0, fit, cb, s, None, iters, 0, ws) for s in range(S)]
    del ws
    sh, ga = shapes.cpu().numpy(), gains.cpu().numpy()
    # the oracle on the same bits: the fit rows of every head, [G][n_fit * M][d], and their token weights
    rows = torch.stack([x[fit[g_], g_] for g_ in range(G)]).float().reshape(G, n_fit * M, d).cpu().numpy()
    w_rows = torch.stack([w[fit[g_]] for g_ in range(G)]).repeat_interleave(M, dim=1).cpu().numpy()
    ref_sh, ref_ga, ref_stats = _oracle_fit_rows(rows, w_rows, K, S, iters, G)
    _assert_fit_matches(sh, ga, stats, ref_sh, ref_ga, ref_stats, G, S)
    # the shapes the fit returns are unit vectors and the gains non-negative (Eq. 3)
    assert np.abs(np.linalg.norm(sh.astype(np.float64), axis=-1) - 1.0).max() <= 1e-6 and (ga >= 0).all()
    # full-cache encode / decode on sampled tokens, against the oracle with ITS codebooks
    shapes.copy_(torch.from_numpy(ref_sh).cuda()); gains.copy_(torch.from_numpy(ref_ga).cuda())
    tok = np.sort(np.random.default_rng(3).choice(T, 2048, replace=False))
    _sampled_encode_decode_check(B, x, view, True, cb, ref_sh, ref_ga, S, tok)


@pytest.mark.parametrize("kind", ["k", "v"])
def test_cfg3_full_size_fit_vs_oracle_and_prefix_sweep(B, kind):
    """BASELINE config 3 at its full size (8 x 32768 x 128, K-like and V-like, S = 4, 20 iterations per stage), bench.py's
    call sequence: the whole fit -> encode trajectory against the oracle (criteria a, b, c, per-iteration J, changed counts),
    the decode of every prefix S = 1..4 of all 2,097,152 rows, and falling weighted residual energy (reading c-N)."""
    dd = inputs.make(3, kind=kind)
    c = dd["config"]
    got, ref = _check_free_running(dd, c.K, c.S, c.iters, "bf16", prefix_encode=True)
    M = c.hd // c.d
    w_rows = np.repeat(dd["w"], M).astype(np.float64)
    energy = [float((w_rows[None] * (o.rows_of(dd["x"], c.d).astype(np.float64) ** 2).sum(-1)).sum())]
    r = o.rows_of(dd["x"], c.d).copy()
    for st in range(c.S):
        for g_ in range(c.G):
            _, r[g_], _, _ = o.encode_stage(r[g_], ref["shapes"][g_, st], ref["gains"][g_, st])
        energy.append(float((w_rows[None] * (r.astype(np.float64) ** 2).sum(-1)).sum()))
    assert all(energy[i + 1] < energy[i] for i in range(c.S))
    for n in range(1, c.S + 1):
        dec = gpu_decode(got["codes_dev"], got["cb"], n, c.G, c.T, c.hd, c.d, dtype="bf16")
        want, _ = o.decode(got["codes"], got["shapes"], got["gains"], c.hd, S_used=n, bf16=True)
        assert np.array_equal(dec, want), n
