"""gsrq_attention_decode_static: the attention step for callers that cannot allocate device memory.

Some users of this library have nowhere to get a workspace from: an inference engine that gave all of the GPU's memory to its KV
cache at start-up, a plug-in that is called while its host is capturing a stream (cudaMalloc / cudaFree are not allowed there, and
outside a capture they stall the whole device), a host process that forbids allocation once it is serving.  For them the library
keeps the split partial results of the attention kernels in a fixed 4 MiB array that is part of the library image
(include/gsrq.h, GSRQ_ATTENTION_STATIC_SCRATCH_BYTES), and gsrq_attention_decode_static takes no workspace at all.

What is checked here, against the existing workspace path gsrq_attention_decode on the same inputs:
  * two calls in a row, of different shapes, so that the second one runs on a buffer that still holds the first one's partial
    results (the buffer is never cleared); then the first shape again;
  * outputs within the tolerance the attention tests use (2e-4 of the largest output magnitude, tests/test_gpu_attention.py) --
    and, since both paths run the same kernels with the same split, bit-equal;
  * a request beyond the buffer is refused with GSRQ_EWORKSPACE before anything is launched;
  * the device's free memory does not shrink across a call once the first call on the device has been made.

This file is named so that pytest collects it last: with `-x` a failure here cannot hide a failure of any other test.  It has to
pass alone in a fresh process (its first call then does the per-device set-up) and after the rest of the suite.  Run with `-m gpu`."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

TOL = 2e-4   # relative to max |out|, as in tests/test_gpu_attention.py


@pytest.fixture(scope="module")
def B():
    import __graft_entry__ as ge
    ge.build()
    from paper_2607_01065_b200 import binding
    return binding


def _inputs(seed, G, Tc, K, SK, SV, Hq, lens):
    """Random codes, codebooks and queries on the device (no oracle involved: the reference is the library's workspace path)."""
    rng = np.random.default_rng(seed)
    hd, d, M = 128, 16, 8
    dev = lambda a: torch.from_numpy(a).cuda()

    def codebook(S, gain):
        s = rng.standard_normal((G, S, K, d))
        s /= np.linalg.norm(s, axis=-1, keepdims=True)
        g = gain * np.abs(rng.standard_normal((G, S, K))) * (0.5 ** np.arange(S))[None, :, None]
        return dev(s.astype(np.float32)), dev(g.astype(np.float32))

    ks, kg = codebook(SK, 3.0)
    vs, vg = codebook(SV, 1.0)
    start = np.concatenate([[0], np.cumsum(lens)[:-1]]).astype(np.int64)
    return dict(q=dev(rng.standard_normal((len(lens), Hq, hd)).astype(np.float32)),
                kc=dev(rng.integers(0, K, (SK, G, Tc * M)).astype(np.uint8)), vc=dev(rng.integers(0, K, (SV, G, Tc * M)).astype(np.uint8)),
                ks=ks, kg=kg, vs=vs, vg=vg, start=dev(start), length=dev(np.array(lens, dtype=np.int64)),
                G=G, SK=SK, SV=SV, rows=Tc * M, max_len=int(max(lens)), hd=hd, d=d)


def _run(B, fn, c, rope_theta, fill):
    out = torch.full((c["q"].shape[0], c["q"].shape[1], c["hd"]), fill, device="cuda")
    fn(c["q"], c["kc"], B.codebook_of(c["ks"], c["kg"]), c["SK"], c["vc"], B.codebook_of(c["vs"], c["vg"]), c["SV"], c["rows"],
       c["start"], c["length"], c["max_len"], c["G"], c["d"], c["hd"] ** -0.5, rope_theta, out)
    torch.cuda.synchronize()
    return out


def _check_same(B, c, rope_theta):
    want = _run(B, B.gsrq_attention_decode, c, rope_theta, 7.0)          # existing path: scratch from a caller-allocated workspace
    got = _run(B, B.gsrq_attention_decode_static, c, rope_theta, -3.0)   # new path: scratch inside the library
    assert torch.isfinite(got).all()
    assert (got - want).abs().max().item() <= TOL * want.abs().max().item()
    assert torch.equal(got, want)   # same kernels, same split of the token range, no atomics
    return got


@pytest.mark.parametrize("rope_theta", [0.0, 500000.0])
def test_static_scratch_path_equals_the_workspace_path_on_calls_in_a_row(B, rope_theta):
    # call 1: several splits per (sequence, KV head), an empty and a one-token sequence, LLaMA-3-8B's 4 query heads per KV head
    big = _inputs(11, G=2, Tc=9000, K=256, SK=2, SV=2, Hq=8, lens=[5000, 0, 3999, 1])
    # call 2: another shape (generic kernel, 8 query heads per KV head, fewer entries) on the buffer call 1 left behind
    small = _inputs(12, G=2, Tc=700, K=100, SK=2, SV=1, Hq=16, lens=[300, 400])
    first = _check_same(B, big, rope_theta)
    _check_same(B, small, rope_theta)
    again = _check_same(B, big, rope_theta)
    assert torch.equal(first, again)
    assert not first[1].any()   # the empty sequence


def test_static_scratch_path_refuses_what_does_not_fit(B):
    cap = B.gsrq_attention_static_scratch_bytes()
    assert cap == 4 << 20
    # 300 sequences x 8 KV heads x 1 split x 4 query heads x 130 floats = 4.99 MB > 4 MiB
    n = 300
    c = _inputs(13, G=8, Tc=n, K=16, SK=1, SV=1, Hq=32, lens=[1] * n)
    launches = B.lib().gsrq_launch_count()
    with pytest.raises(B.GsrqError) as e:
        _run(B, B.gsrq_attention_decode_static, c, 0.0, 5.0)
    assert e.value.code == -3 and "4194304" in str(e.value)   # GSRQ_EWORKSPACE, with the buffer size in the message
    assert B.lib().gsrq_launch_count() == launches            # nothing was launched
    # 252 sequences is the largest batch of this head configuration that fits (include/gsrq.h)
    c = _inputs(14, G=8, Tc=252, K=16, SK=1, SV=1, Hq=32, lens=[1] * 252)
    _check_same(B, c, 0.0)


def test_static_scratch_path_takes_no_device_memory(B):
    c = _inputs(15, G=8, Tc=4096, K=256, SK=2, SV=2, Hq=32, lens=[4096])
    out = torch.empty(1, 32, 128, device="cuda")
    call = lambda: B.gsrq_attention_decode_static(c["q"], c["kc"], B.codebook_of(c["ks"], c["kg"]), 2, c["vc"], B.codebook_of(c["vs"], c["vg"]), 2,
                                                  c["rows"], c["start"], c["length"], c["max_len"], 8, 16, 128 ** -0.5, 0.0, out)
    call()   # per-device set-up and the kernels' code are in place after this
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        call()
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, (free0, free1)
