"""The host-buffer entry points and the boundary's argument checks on a real device (`-m gpu`):
gsrq_pipeline_host (fit on all tokens, and on a token subset) must return exactly what the step-wise device calls
return; a degenerate group and a misaligned tensor pointer are reported as error codes, not as faults."""
import numpy as np
import pytest
import torch

from paper_2607_01065_b200.pipeline import gpu_decode, gpu_gsrq
from paper_2607_01065_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import __graft_entry__ as ge
    ge.build()
    from paper_2607_01065_b200 import binding
    return binding


@pytest.mark.parametrize("subset", [False, True])
def test_pipeline_host_equals_stepwise_device_calls(B, subset):
    dd = inputs.make(1, T=640)
    c = dd["config"]
    K, S, iters = 128, 2, 5
    fit = inputs.fit_sample(c.G, 640, 200, 77) if subset else None
    ref = gpu_gsrq(dd["x"], dd["w"], c.d, K, S, iters, dtype="bf16", fit_tokens=fit, pass_residual=not subset, prefix_encode=not subset,
                   want_residual=False)
    dec = gpu_decode(ref["codes_dev"], ref["cb"], S, c.G, 640, c.hd, c.d, dtype="bf16")
    x_h = torch.from_numpy(dd["x"]).to(torch.bfloat16).pin_memory()
    w_h = torch.from_numpy(dd["w"]).pin_memory()
    fit_h = None if fit is None else torch.from_numpy(fit)
    M = c.hd // c.d
    sh_h = torch.empty(c.G, S, K, c.d); ga_h = torch.empty(c.G, S, K)
    co_h = torch.empty(S, c.G, 640 * M, dtype=torch.uint8); out_h = torch.empty(c.G, 640, c.hd, dtype=torch.bfloat16)
    view = B.view_of(x_h, c.d)
    for _ in range(2):   # the second call reuses the library's private pool
        B.gsrq_pipeline_host(x_h, view, w_h, fit_h, K, S, iters, 0, sh_h, ga_h, co_h, out_h)
        assert np.array_equal(sh_h.numpy(), ref["shapes"]) and np.array_equal(ga_h.numpy(), ref["gains"])
        assert np.array_equal(co_h.numpy(), ref["codes"])
        assert np.array_equal(out_h.float().numpy(), dec)
    B.gsrq_release_host_pool()


def test_pipeline_host_reports_a_degenerate_group(B):
    x_h = torch.zeros(2, 64, 128, dtype=torch.bfloat16)
    x_h[0] = torch.randn(64, 128).to(torch.bfloat16)        # group 0 is fine, group 1 is all zeros
    K, S = 16, 1
    sh_h = torch.empty(2, S, K, 16); ga_h = torch.empty(2, S, K); co_h = torch.empty(S, 2, 64 * 8, dtype=torch.uint8)
    with pytest.raises(B.GsrqError) as e:
        B.gsrq_pipeline_host(x_h, B.view_of(x_h, 16), None, None, K, S, 3, 0, sh_h, ga_h, co_h, None)
    assert e.value.code == -5


def test_pipeline_host_batch_equals_single_calls(B):
    """Three tensors (K-like, V-like, K-like) in one pipelined call over two streams: bit-identical to three gsrq_pipeline_host calls;
    the third tensor reuses the first one's stream.  One of them without decode output."""
    c = inputs.CONFIGS[1]
    T, K, S, iters = 1024, 256, 2, 4
    xs = [inputs.k_like(c.G, T, c.hd, 901), inputs.v_like(c.G, T, c.hd, 902), inputs.k_like(c.G, T, c.hd, 903)]
    w = inputs.token_weights(T, 904)
    fit = inputs.fit_sample(c.G, T, 300, 905)
    M = c.hd // c.d
    x_h = [torch.from_numpy(x).to(torch.bfloat16).pin_memory() for x in xs]
    w_h = torch.from_numpy(w).pin_memory(); fit_h = torch.from_numpy(fit).pin_memory()
    view = B.view_of(x_h[0], c.d)
    mk = lambda: (torch.empty(c.G, S, K, c.d).pin_memory(), torch.empty(c.G, S, K).pin_memory(),
                  torch.empty(S, c.G, T * M, dtype=torch.uint8).pin_memory(), torch.empty(c.G, T, c.hd, dtype=torch.bfloat16).pin_memory())
    single = [mk() for _ in xs]
    for x, (sh, ga, co, out) in zip(x_h, single):
        B.gsrq_pipeline_host(x, view, w_h, fit_h, K, S, iters, 0, sh, ga, co, out)
    batch = [mk() for _ in xs]
    B.gsrq_pipeline_host_batch(x_h, view, [w_h] * 3, [fit_h] * 3, K, S, iters, 0, [b[0] for b in batch], [b[1] for b in batch], [b[2] for b in batch],
                               [batch[0][3], None, batch[2][3]])
    for i, (s_, b_) in enumerate(zip(single, batch)):
        assert torch.equal(s_[0], b_[0]) and torch.equal(s_[1], b_[1]) and torch.equal(s_[2], b_[2]), i
        if i != 1:
            assert torch.equal(s_[3], b_[3]), i
    # a degenerate tensor in the middle is reported, the others are still processed
    bad = torch.zeros_like(x_h[1])
    with pytest.raises(B.GsrqError) as e:
        B.gsrq_pipeline_host_batch([x_h[0], bad, x_h[2]], view, None, None, K, S, 2, 0, [b[0] for b in batch], [b[1] for b in batch],
                                   [b[2] for b in batch], None)
    assert e.value.code == -5
    B.gsrq_release_host_pool()


def test_misaligned_tensor_pointer_is_an_error_not_a_fault(B):
    buf = torch.zeros(2 * 64 * 128 + 8, dtype=torch.bfloat16, device="cuda")
    x = buf[4:4 + 2 * 64 * 128].view(2, 64, 128)            # base offset by 8 bytes
    assert x.data_ptr() % 16 == 8
    view = B.view_of(x, 16)
    sh = torch.zeros(2, 1, 16, 16, device="cuda"); ga = torch.zeros(2, 1, 16, device="cuda")
    cb = B.codebook_of(sh, ga)
    ws = B.workspace(view, 16, 1, 0)
    codes = torch.zeros(1, 2, 64 * 8, dtype=torch.uint8, device="cuda")
    for call in (lambda: B.gsrq_fit_stage(x, view, None, 0, None, cb, 0, None, 2, 0, ws),
                 lambda: B.gsrq_encode(x, view, cb, 0, 1, codes, None, ws),
                 lambda: B.gsrq_decode(codes, cb, 1, x, view)):
        with pytest.raises(B.GsrqError) as e:
            call()
        assert e.value.code == -1
    torch.cuda.synchronize()                                 # no sticky fault was raised
