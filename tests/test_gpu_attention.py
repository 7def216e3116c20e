"""Decode fused into attention (gsrq_attention_decode; PAPER.md:443 (ii)) against the fp64 oracle (oracle/attn_oracle.py): GQA over
GSRQ codes with and without the rotary embedding, several sequences of different lengths, split over CTAs.  Floating point:
the kernel works in fp32 (logits of magnitude <= ~30, sums over <= 10^5 terms), so outputs agree with the fp64 oracle to
2e-4 relative to the output's largest magnitude (derivation: DESIGN.md, attention row).  Run with `-m gpu` on a B200."""
import numpy as np
import pytest
import torch

from oracle import attn_oracle as ao

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import __graft_entry__ as ge
    ge.build()
    from paper_2607_01065_b200 import binding
    return binding


def _case(seed, G, Tc, K, SK, SV, Bq, Hq, d=16):
    rng = np.random.default_rng(seed)
    hd = 128
    M = hd // d
    def cb(S, gain):
        s = rng.standard_normal((G, S, K, d)); s /= np.linalg.norm(s, axis=-1, keepdims=True)
        g = (gain * np.abs(rng.standard_normal((G, S, K))) * (0.5 ** np.arange(S))[None, :, None])
        return s.astype(np.float32), g.astype(np.float32)
    ks, kg = cb(SK, 3.0); vs, vg = cb(SV, 1.0)
    kc = rng.integers(0, K, (SK, G, Tc * M)).astype(np.uint8)
    vc = rng.integers(0, K, (SV, G, Tc * M)).astype(np.uint8)
    q = rng.standard_normal((Bq, Hq, hd)).astype(np.float32)
    return dict(ks=ks, kg=kg, vs=vs, vg=vg, kc=kc, vc=vc, q=q, G=G, Tc=Tc, hd=hd, d=d, M=M)


@pytest.mark.parametrize("rope_theta", [0.0, 500000.0])
@pytest.mark.parametrize("G,Tc,K,SK,SV,Hq,lens", [
    (2, 9000, 256, 2, 2, 8, [5000, 0, 3999, 1]),      # GQA 4:1 (LLaMA-3-8B's ratio), an empty and a one-token sequence, several splits
    (1, 3000, 100, 1, 3, 1, [3000]),                   # single head, K < 256, different stage counts for keys and values
    (2, 700, 256, 4, 1, 8, [300, 400]),                # 4 key stages, 1 value stage (generic kernel)
    (2, 600, 256, 2, 2, 16, [200, 400]),               # 8 query heads per KV head
])
def test_attention_decode_matches_oracle(B, rope_theta, G, Tc, K, SK, SV, Hq, lens):
    Bq = len(lens)
    c = _case(7 + Tc, G, Tc, K, SK, SV, Bq, Hq)
    start = np.concatenate([[0], np.cumsum(lens)[:-1]]).astype(np.int64)
    length = np.array(lens, dtype=np.int64)
    want = ao.attention_decode(c["q"], c["kc"], c["ks"], c["kg"], c["vc"], c["vs"], c["vg"], c["hd"], start, length, rope_theta=rope_theta)
    dev = lambda a: torch.from_numpy(a).cuda()
    ks, kg, vs, vg = dev(c["ks"]), dev(c["kg"]), dev(c["vs"]), dev(c["vg"])
    out = torch.full((Bq, Hq, c["hd"]), 7.0, device="cuda")
    B.gsrq_attention_decode(dev(c["q"]), dev(c["kc"]), B.codebook_of(ks, kg), SK, dev(c["vc"]), B.codebook_of(vs, vg), SV, Tc * c["M"],
                            dev(start), dev(length), int(max(lens)), G, c["d"], 1.0 / np.sqrt(c["hd"]), rope_theta, out)
    torch.cuda.synchronize()
    got = out.cpu().numpy().astype(np.float64)
    scale = np.abs(want).max()
    assert np.abs(got - want).max() <= 2e-4 * scale, np.abs(got - want).max() / scale
    for b, n in enumerate(lens):
        if n == 0:
            assert not got[b].any()
    # run-to-run bit identity (no atomics)
    out2 = torch.zeros_like(out)
    B.gsrq_attention_decode(dev(c["q"]), dev(c["kc"]), B.codebook_of(ks, kg), SK, dev(c["vc"]), B.codebook_of(vs, vg), SV, Tc * c["M"],
                            dev(start), dev(length), int(max(lens)), G, c["d"], 1.0 / np.sqrt(c["hd"]), rope_theta, out2)
    assert torch.equal(out, out2)


def test_attention_on_an_encoded_cache_equals_attention_on_the_decoded_tensor(B):
    """End to end on the library's own codes: fit + encode a K-like and a V-like cache, then attention from the codes equals
    plain attention on gsrq_decode's fp32 output."""
    from paper_2607_01065_b200.pipeline import gpu_gsrq
    from paper_2607_01065_b200 import inputs
    G, T, hd, d, K, S = 2, 1024, 128, 16, 256, 2
    xk = inputs.k_like(G, T, hd, 777); xv = inputs.v_like(G, T, hd, 778)
    w = inputs.token_weights(T, 779)
    gk = gpu_gsrq(xk, w, d, K, S, 4, dtype="bf16", prefix_encode=True)
    gv = gpu_gsrq(xv, w, d, K, S, 4, dtype="bf16", prefix_encode=True)
    q = torch.randn(1, 8, hd, device="cuda", generator=torch.Generator(device="cuda").manual_seed(1))
    start = torch.zeros(1, dtype=torch.int64, device="cuda"); length = torch.full((1,), T, dtype=torch.int64, device="cuda")
    out = torch.zeros(1, 8, hd, device="cuda")
    B.gsrq_attention_decode(q, gk["codes_dev"], gk["cb"], S, gv["codes_dev"], gv["cb"], S, T * 8, start, length, T, G, d, hd ** -0.5, 0.0, out)
    kd = torch.zeros(G, T, hd, device="cuda"); vd = torch.zeros(G, T, hd, device="cuda")
    B.gsrq_decode(gk["codes_dev"], gk["cb"], S, kd, B.view_of(kd, d))
    B.gsrq_decode(gv["codes_dev"], gv["cb"], S, vd, B.view_of(vd, d))
    want = torch.nn.functional.scaled_dot_product_attention(q.double().view(1, G, 4, hd), kd.double()[None], vd.double()[None]).view(1, 8, hd)
    assert (out.double() - want).abs().max() <= 2e-4 * want.abs().max()


def test_attention_sequence_outside_the_code_planes_is_served_as_empty(B):
    """A (seq_start, seq_len) pair that reaches beyond plane_rows / 8 tokens is never read: its output rows are zeros, the other
    sequences of the call are unaffected (include/gsrq.h)."""
    G, Tc, K, S, Hq = 2, 300, 256, 2, 8
    c = _case(91, G, Tc, K, S, S, 3, Hq)
    start = np.array([0, 200, -1], dtype=np.int64); length = np.array([300, 200, 10], dtype=np.int64)
    want = ao.attention_decode(c["q"][:1], c["kc"], c["ks"], c["kg"], c["vc"], c["vs"], c["vg"], c["hd"], start[:1], length[:1], rope_theta=0.0)
    dev = lambda a: torch.from_numpy(a).cuda()
    ks, kg, vs, vg = dev(c["ks"]), dev(c["kg"]), dev(c["vs"]), dev(c["vg"])
    for fn in (B.gsrq_attention_decode, B.gsrq_attention_decode_static):
        out = torch.full((3, Hq, c["hd"]), 7.0, device="cuda")
        fn(dev(c["q"]), dev(c["kc"]), B.codebook_of(ks, kg), S, dev(c["vc"]), B.codebook_of(vs, vg), S, Tc * c["M"], dev(start), dev(length),
           300, G, c["d"], 1.0 / np.sqrt(c["hd"]), 0.0, out)
        got = out.cpu().numpy().astype(np.float64)
        assert np.abs(got[0] - want[0]).max() <= 2e-4 * np.abs(want).max()
        assert not got[1:].any()


@pytest.mark.parametrize("rope_theta", [0.0, 500000.0])
@pytest.mark.parametrize("G,Tc,K,SK,SV,Hq,lens", [
    (2, 2500, 256, 12, 12, 8, [1500, 0, 999, 1]),    # the paper's point: D = 128, R = 12 (0.75 bits per element), GQA 4:1
    (1, 700, 100, 16, 32, 8, [700]),                 # R = 16 keys, R = 32 values, K < 256, 8 query heads on one KV head
    (2, 300, 256, 1, 3, 2, [120, 180]),              # one query head per KV head, few stages
])
def test_attention_decode_at_the_papers_operating_point_matches_oracle(B, rope_theta, G, Tc, K, SK, SV, Hq, lens):
    """d = head_dim = 128 (one sub-vector per token and head), up to 32 stages: the configuration the paper's latency tables are
    measured at, against the same fp64 oracle and with the same 2e-4 tolerance (reading a-T) as d = 16."""
    Bq = len(lens)
    c = _case(300 + Tc, G, Tc, K, SK, SV, Bq, Hq, d=128)
    start = np.concatenate([[0], np.cumsum(lens)[:-1]]).astype(np.int64)
    length = np.array(lens, dtype=np.int64)
    want = ao.attention_decode(c["q"], c["kc"], c["ks"], c["kg"], c["vc"], c["vs"], c["vg"], c["hd"], start, length, rope_theta=rope_theta)
    dev = lambda a: torch.from_numpy(a).cuda()
    ks, kg, vs, vg = dev(c["ks"]), dev(c["kg"]), dev(c["vs"]), dev(c["vg"])
    outs = []
    for _ in range(2):
        out = torch.full((Bq, Hq, c["hd"]), 7.0, device="cuda")
        B.gsrq_attention_decode(dev(c["q"]), dev(c["kc"]), B.codebook_of(ks, kg), SK, dev(c["vc"]), B.codebook_of(vs, vg), SV, Tc * c["M"],
                                dev(start), dev(length), int(max(lens)), G, c["d"], 1.0 / np.sqrt(c["hd"]), rope_theta, out)
        outs.append(out)
    got = outs[0].cpu().numpy().astype(np.float64)
    scale = np.abs(want).max()
    assert np.abs(got - want).max() <= 2e-4 * scale, np.abs(got - want).max() / scale
    for b, n in enumerate(lens):
        if n == 0:
            assert not got[b].any()
    assert torch.equal(outs[0], outs[1])   # run-to-run bit identity
