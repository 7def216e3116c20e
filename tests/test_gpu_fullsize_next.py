"""The rows SURVEY.md section 8 lists after the headline path, at the sizes and in the launch configurations bench.py times
(`extras.d128`, `extras.attention_decode`), against the CPU oracle on sampled outputs it can compute one by one:

* D = 128, K = 256, R = 12 stages on a K-like 8 x 32768 x 128 bf16 layer.  The 12 full-size fits are out of the
  oracle's reach (10^12 fp64 multiply-adds), so: (a) one full-size Lloyd iteration of stage 0 is compared codebook by codebook on
  two heads; (b) with the GPU's 12 codebooks, the codes / residual / decoded values of sampled rows (a fixed-codebook encode is
  per row) including the last tile's.
* decode-attention at batch 8 x 131,072 tokens, 32 query / 8 KV heads, S = 2 (PAPER.md:443 (ii), 457-473): the whole launch on the
  GPU, the fp64 oracle on two (sequence, KV head) pairs.

Run with `-m gpu` on a B200."""
import numpy as np
import pytest
import torch

from paper_2607_01065_b200.pipeline import gpu_decode, gpu_gsrq, stats_np, to_device
from oracle import attn_oracle as ao
from oracle import gsrq_oracle as o
from paper_2607_01065_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import __graft_entry__ as ge
    ge.build()
    from paper_2607_01065_b200 import binding
    return binding


def test_d128_bench_size_one_full_lloyd_iteration(B):
    G, T, hd, d, K = 8, 32768, 128, 128, 256
    x_np = inputs.k_like(G, T, hd, inputs.seed_of(3, "k"))
    w_np = inputs.token_weights(T, inputs.seed_of(3, "w"))
    x = to_device(x_np, "bf16")
    view = B.view_of(x, d)
    shapes = torch.zeros(G, 1, K, d, device="cuda"); gains = torch.zeros(G, 1, K, device="cuda")
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, 1, 0)
    st = B.gsrq_fit_stage(x, view, torch.from_numpy(w_np).cuda(), 0, None, cb, 0, None, 1, 0, ws)
    torch.cuda.synchronize()
    rows = o.rows_of(x_np, d)
    for g_ in (0, 5):
        ref = o.fit_stage(rows[g_], w_np, K, 1, seed=0, group=g_, G=G, stage=0)
        assert np.abs(shapes[g_, 0].cpu().numpy() - ref["shapes"]).max() <= 1e-6
        assert np.abs(gains[g_, 0].cpu().numpy() - ref["gains"]).max() <= 1e-5
        s_got = stats_np(st, g_)
        assert s_got["iters_run"] == ref["iters_run"]
        np.testing.assert_allclose(s_got["J"], ref["J_assign"], rtol=1e-4)
        assert np.array_equal(s_got["changed"], ref["changed"])


def test_d128_bench_size_sampled_encode_decode(B):
    G, T, hd, d, K, S, iters = 8, 32768, 128, 128, 256, 12, 10
    x_np = inputs.k_like(G, T, hd, inputs.seed_of(3, "k"))
    w_np = inputs.token_weights(T, inputs.seed_of(3, "w"))
    got = gpu_gsrq(x_np, w_np, d, K, S, iters, seed=0, dtype="bf16", prefix_encode=True)   # bench.py's fit_all
    rng = np.random.default_rng(11)
    tok = np.unique(np.concatenate([rng.choice(T, 1200, replace=False), np.arange(T - 130, T), np.arange(0, 40)]))
    codes_o, res_o, _, _ = o.encode(x_np[:, tok], got["shapes"], got["gains"], d)
    assert np.array_equal(got["codes"][:, :, tok], codes_o)
    assert np.array_equal(got["residual"][:, tok], res_o.reshape(G, len(tok), d))
    for n in (1, 8, 12):                    # 1/16, 1/2, 3/4 bit per element
        dec = gpu_decode(got["codes_dev"], got["cb"], n, G, T, hd, d, dtype="bf16")
        want, _ = o.decode(codes_o[:n], got["shapes"][:, :n], got["gains"][:, :n], hd, bf16=True)
        assert np.array_equal(dec[:, tok], want), n
    # what 12 stages leave of the layer's energy (RQ): bench.py reports 0.10 for this layer
    assert float((got["residual"].astype(np.float64) ** 2).sum()) < 0.25 * float((x_np.astype(np.float64) ** 2).sum())


@pytest.mark.parametrize("rope_theta", [0.0, 500000.0])
def test_attention_bench_size_sampled(B, rope_theta):
    G, Hq, hd, d, K, S, Bq, ctx, M = 8, 32, 128, 16, 256, 2, 8, 131072, 8
    n_rep = Hq // G
    rng = np.random.default_rng(2024)
    T = Bq * ctx
    kc = rng.integers(0, K, (S, G, T * M), dtype=np.uint8)
    vc = rng.integers(0, K, (S, G, T * M), dtype=np.uint8)

    def cb(gain):
        s = rng.standard_normal((G, S, K, d)); s /= np.linalg.norm(s, axis=-1, keepdims=True)
        g = gain * np.abs(rng.standard_normal((G, S, K))) * (0.5 ** np.arange(S))[None, :, None]
        return s.astype(np.float32), g.astype(np.float32)
    ks, kg = cb(3.0); vs, vg = cb(1.0)
    q = rng.standard_normal((Bq, Hq, hd)).astype(np.float32)
    dev = lambda a: torch.from_numpy(a).cuda()
    start = torch.arange(Bq, dtype=torch.int64, device="cuda") * ctx
    length = torch.full((Bq,), ctx, dtype=torch.int64, device="cuda")
    out = torch.zeros(Bq, Hq, hd, device="cuda")
    ksd, kgd, vsd, vgd = dev(ks), dev(kg), dev(vs), dev(vg)
    B.gsrq_attention_decode(dev(q), dev(kc), B.codebook_of(ksd, kgd), S, dev(vc), B.codebook_of(vsd, vgd), S, T * M, start, length, ctx, G, d,
                            hd ** -0.5, rope_theta, out)
    torch.cuda.synchronize()
    got = out.cpu().numpy().astype(np.float64)
    for b, g_ in ((0, 0), (7, 5)):
        sl = slice(b * ctx * M, (b + 1) * ctx * M)
        want = ao.attention_decode(q[b:b + 1, g_ * n_rep:(g_ + 1) * n_rep], kc[:, g_:g_ + 1, sl], ks[g_:g_ + 1], kg[g_:g_ + 1],
                                   vc[:, g_:g_ + 1, sl], vs[g_:g_ + 1], vg[g_:g_ + 1], hd, np.zeros(1, np.int64), np.full(1, ctx, np.int64),
                                   rope_theta=rope_theta)
        diff = np.abs(got[b, g_ * n_rep:(g_ + 1) * n_rep] - want[0]).max()
        assert diff <= 2e-4 * np.abs(want).max(), (b, g_, diff / np.abs(want).max())
