"""Variants around the encoder on the GPU against oracle/variants_oracle.py: log-smoothed gradient weights
(PAPER.md:192 Eq. 9, :434 Eq. 10), per-vector fp16 gain codes, nibble packing, per-subspace codebooks.
Run with `-m gpu` on a B200."""
import numpy as np
import pytest
import torch

from paper_2607_01065_b200.pipeline import gpu_gsrq, to_device
from oracle import gsrq_oracle as o
from oracle import variants_oracle as vo
from paper_2607_01065_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import __graft_entry__ as ge
    ge.build()
    from paper_2607_01065_b200 import binding
    return binding


@pytest.mark.parametrize("T,dtype", [(4097, "f32"), (6000, "bf16")])
def test_log_weights(B, T, dtype):
    rng = np.random.default_rng(T)
    G, hd = 3, 128
    g = (rng.standard_normal((G, T, hd)) * np.exp(1.5 * rng.standard_normal((G, T, 1)))).astype(np.float32)   # heavy-tailed norms
    if dtype == "bf16":
        g = inputs.bf16_round(g)
    x = to_device(g, dtype)
    view = B.view_of(x, 16)
    w = torch.zeros(G, T, device="cuda")
    B.gsrq_log_weights(x, view, 1.0, 1e-12, w)
    torch.cuda.synchronize()
    want = vo.log_weights(g, 1.0, 1e-12)
    np.testing.assert_allclose(w.cpu().numpy(), want, rtol=2e-6, atol=1e-7)
    nrm = np.linalg.norm(g.astype(np.float64), axis=-1)
    assert (nrm.max(1) / np.median(nrm, 1)).min() > 50 and (want.max(1) / np.median(want, 1)).max() < 10    # the compression PAPER.md:196 describes


@pytest.mark.parametrize("d,K,S,dtype", [(16, 256, 2, "bf16"), (8, 16, 3, "f32"), (32, 64, 2, "bf16")])
def test_pervector_gain_codes(B, d, K, S, dtype):
    G, T, hd = 2, 777, 128 if d != 8 else 8
    x_np = inputs.k_like(G, T, hd, 900 + d) if hd == 128 else np.stack([inputs.tiny(900 + g_, T, 8)[0] for g_ in range(G)])
    if dtype == "bf16":
        x_np = inputs.bf16_round(x_np)
    rows = o.rows_of(x_np, d)
    rng = np.random.default_rng(d)
    s_np = rng.standard_normal((G, S, K, d)); s_np = (s_np / np.linalg.norm(s_np, axis=-1, keepdims=True)).astype(np.float32)
    x = to_device(x_np, dtype)
    view = B.view_of(x, d)
    M = hd // d
    N = T * M
    shapes = torch.from_numpy(s_np).cuda(); gains = torch.ones(G, S, K, device="cuda")
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, S, 0)
    codes = torch.zeros(S, G, N, dtype=torch.uint8, device="cuda")
    g16 = torch.zeros(S, G, N, dtype=torch.float16, device="cuda")
    res = torch.zeros(G, N, d, device="cuda")
    B.gsrq_encode_pervector_gain(x, view, cb, S, codes, g16, res, ws)
    out = torch.zeros_like(x)
    B.gsrq_decode_pervector_gain(codes, g16, cb, S, out, view)
    torch.cuda.synchronize()
    for g_ in range(G):
        r = rows[g_]
        cs, gs = [], []
        for st in range(S):
            c, gam, r = vo.encode_stage_pervector_gain(r, s_np[g_, st])
            cs.append(c); gs.append(gam)
            assert np.array_equal(codes[st, g_].cpu().numpy(), c), (g_, st)
            assert np.array_equal(g16[st, g_].cpu().numpy(), gam), (g_, st)
        assert np.array_equal(res[g_].cpu().numpy(), r)
        xhat = vo.decode_pervector_gain(np.stack(cs), np.stack(gs), s_np[g_])
        want = inputs.bf16_round(xhat) if dtype == "bf16" else xhat
        assert np.array_equal(out[g_].float().cpu().numpy().reshape(N, d), want)


def test_nibble_packing(B):
    rng = np.random.default_rng(5)
    c = rng.integers(0, 16, (6, 4097)).astype(np.uint8)
    cd = torch.from_numpy(c).cuda()
    packed = torch.zeros(6, 2049, dtype=torch.uint8, device="cuda")
    B.gsrq_pack_nibbles(cd, 16, 6, 4097, packed)
    with pytest.raises(B.GsrqError) as e:   # K > 16: a code would lose its high bits
        B.gsrq_pack_nibbles(cd, 17, 6, 4097, packed)
    assert e.value.code == -1
    assert np.array_equal(packed.cpu().numpy(), vo.pack_nibbles(c))
    back = torch.zeros_like(cd)
    B.gsrq_unpack_nibbles(packed, 6, 4097, back)
    assert torch.equal(back, cd)
    # cfg 0 of BASELINE.json: K = 16 codes of the tiny sanity config survive the 4-bit storage
    dd = inputs.make(0)
    cfg = dd["config"]
    got = gpu_gsrq(dd["x"], dd["w"], cfg.d, cfg.K, cfg.S, cfg.iters, seed=0, dtype="f32")
    n = got["codes"].shape[-1]
    pk = torch.zeros(cfg.S * cfg.G, (n + 1) // 2, dtype=torch.uint8, device="cuda")
    B.gsrq_pack_nibbles(got["codes_dev"], cfg.K, cfg.S * cfg.G, n, pk)
    un = torch.zeros_like(got["codes_dev"])
    B.gsrq_unpack_nibbles(pk, cfg.S * cfg.G, n, un)
    assert torch.equal(un, got["codes_dev"]) and pk.numel() * 2 == got["codes_dev"].numel()


def test_per_subspace_codebooks(B):
    """an independent codebook per subspace.  Subspace m of a [G][T][hd] tensor is the view {G, T, hd' = d} on the pointer
    shifted by m d elements; a head-inner [T][G][hd] tensor is one view with G M groups.  Both equal the oracle run per subspace."""
    G, T, hd, d, K, S, iters = 2, 600, 128, 16, 64, 2, 4
    M = hd // d
    x_np = inputs.v_like(G, T, hd, 950)
    w_np = inputs.token_weights(T, 951)
    x = to_device(x_np, "bf16")
    for m in (0, 5):
        sub = x[:, :, m * d:(m + 1) * d]                      # a strided slice: same strides, hd' = d
        view = B.gsrq_view(B.GSRQ_BF16, G, T, d, d, x.stride(0), x.stride(1))
        shapes = torch.zeros(G, S, K, d, device="cuda"); gains = torch.zeros(G, S, K, device="cuda")
        cb = B.codebook_of(shapes, gains)
        ws = B.workspace(view, K, S, 0)
        codes = torch.zeros(S, G, T, dtype=torch.uint8, device="cuda")
        res = torch.zeros(G, T, d, device="cuda")
        w = torch.from_numpy(w_np).cuda()
        for st in range(S):
            B.gsrq_fit_stage(sub, view, w, 0, None, cb, st, res if st else None, iters, 0, ws, want_stats=False)
            B.gsrq_encode(sub, view, cb, 0, st + 1, codes, res, ws)
        torch.cuda.synchronize()
        ref = o.gsrq_fit_encode(np.ascontiguousarray(x_np[:, :, m * d:(m + 1) * d]), w_np, d, K, S, iters, seed=0)
        assert np.array_equal(codes.cpu().numpy(), ref["codes"]) and np.abs(shapes.cpu().numpy() - ref["shapes"]).max() <= 1e-6
    # head-inner: one call, G * M groups (group index g * M + m)
    xi = x.permute(1, 0, 2).contiguous()                       # [T][G][hd]
    view = B.gsrq_view(B.GSRQ_BF16, G * M, T, d, d, d, G * hd)
    shapes = torch.zeros(G * M, 1, K, d, device="cuda"); gains = torch.zeros(G * M, 1, K, device="cuda")
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, 1, 0)
    B.gsrq_fit_stage(xi, view, torch.from_numpy(w_np).cuda(), 0, None, cb, 0, None, iters, 0, ws, want_stats=False)
    torch.cuda.synchronize()
    flat = np.ascontiguousarray(x_np.reshape(G, T, M, d).transpose(0, 2, 1, 3).reshape(G * M, T, d))
    ref = o.gsrq_fit_encode(flat, w_np, d, K, 1, iters, seed=0, encode=False)
    assert np.abs(shapes.cpu().numpy() - ref["shapes"]).max() <= 1e-6 and np.abs(gains.cpu().numpy() - ref["gains"]).max() <= 1e-5


def test_code_bytes_beyond_K_are_clamped_not_followed(B):
    """Caller-supplied code bytes >= K (possible when K < 256) must not index past the codebook: the cold decode paths clamp them
    to K - 1 (d = 8 generic kernel, d = 64 wide kernel, per-vector-gain decode)."""
    rng = np.random.default_rng(17)
    for d, hd in ((8, 32), (64, 128)):
        G, T, K, S = 2, 37, 5, 2
        M = hd // d
        sh = rng.standard_normal((G, S, K, d)).astype(np.float32); sh /= np.linalg.norm(sh, axis=-1, keepdims=True)
        gn = np.abs(rng.standard_normal((G, S, K))).astype(np.float32)
        codes = rng.integers(0, K, (S, G, T * M)).astype(np.uint8)
        wild = codes.copy(); wild[codes == K - 1] = 255
        shd, gnd = torch.from_numpy(sh).cuda(), torch.from_numpy(gn).cuda()
        cb = B.codebook_of(shd, gnd)
        a = torch.zeros(G, T, hd, device="cuda"); b = torch.full_like(a, 3.0)
        B.gsrq_decode(torch.from_numpy(codes).cuda(), cb, S, a, B.view_of(a, d))
        B.gsrq_decode(torch.from_numpy(wild).cuda(), cb, S, b, B.view_of(b, d))
        assert torch.equal(a, b)
        if d == 8:
            g16 = torch.from_numpy(np.abs(rng.standard_normal((S, G, T * M))).astype(np.float16)).cuda()
            B.gsrq_decode_pervector_gain(torch.from_numpy(codes).cuda(), g16, cb, S, a, B.view_of(a, d))
            B.gsrq_decode_pervector_gain(torch.from_numpy(wild).cuda(), g16, cb, S, b, B.view_of(b, d))
            assert torch.equal(a, b)
