"""Tensor-core (tcgen05) scoring filter: raw scores vs exact arithmetic, and the validity of its
error bound E_i.  Run with `-m gpu` on a B200."""
import numpy as np
import pytest
import torch

from paper_2607_01065_b200.pipeline import to_device
from oracle import gsrq_oracle as o
from paper_2607_01065_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import __graft_entry__ as ge
    ge.build()
    from paper_2607_01065_b200 import binding
    return binding


def _codebook(rows, K, seed, w=None):
    f = o.fit_stage(rows, w, K, 3, seed=seed)
    return f["shapes"], f["gains"]


@pytest.mark.parametrize("kind,T,K,use_residual", [("k", 200, 256, False), ("v", 131, 256, False),
                                                   ("k", 96, 100, False), ("k", 150, 256, True)])
def test_tc_scores_match_exact_within_bound(B, kind, T, K, use_residual):
    dd = inputs.make(1 if kind == "k" else 2, kind=kind, T=T)
    c = dd["config"]
    G, d, M = 2, c.d, c.hd // c.d
    x_np = dd["x"][:G]
    rows = o.rows_of(x_np, d)
    s_np = np.zeros((G, 1, K, d), np.float32); g_np = np.zeros((G, 1, K), np.float32)
    res_np = None
    if use_residual:                       # fp32 (not bf16-exact) rows: the A operand is split hi + lo
        res_np = rows.copy()
        for g_ in range(G):
            s0, g0 = _codebook(rows[g_], 64, 1)
            _, res_np[g_], _, _ = o.encode_stage(rows[g_], s0, g0)
        rows = res_np
    for g_ in range(G):
        s_np[g_, 0], g_np[g_, 0] = _codebook(rows[g_], K, 0)
    x = to_device(x_np, "bf16")
    view = B.view_of(x, d)
    res = None if res_np is None else torch.from_numpy(res_np).cuda()
    shapes, gains = torch.from_numpy(s_np).cuda(), torch.from_numpy(g_np).cuda()
    cb = B.codebook_of(shapes, gains)
    ws = B.workspace(view, K, 1, 0)
    N = rows.shape[1]
    for mode in (0, 1):
        scores = torch.zeros(G, N, 256, device="cuda")
        idx = torch.zeros(G, N, dtype=torch.uint8, device="cuda")
        B.gsrq_debug_scores(x, view, res, cb, 0, mode, scores, idx, ws)
        torch.cuda.synchronize()
        sc = scores.cpu().numpy().astype(np.float64)
        for g_ in range(G):
            r64, s64, g64 = rows[g_].astype(np.float64), s_np[g_, 0].astype(np.float64), g_np[g_, 0].astype(np.float64)
            dots = r64 @ s64.T
            exact = 2 * g64[None] * dots - g64[None] ** 2 if mode == 0 else 2 * dots
            err = np.abs(sc[g_][:, :K] - exact)
            nrm = np.linalg.norm(r64, axis=1)
            gm = g64.max() if mode == 0 else 1.0
            rho = (4.0 if use_residual else 1.5) * 2.0 ** -17
            E = rho * 2 * gm * nrm + (2.0 ** -20 * gm * gm if mode == 0 else 0.0)
            ratio = (err / np.maximum(E[:, None], 1e-30)).max()
            print(f"tc filter error / bound: {ratio:.3f} (kind={kind} K={K} residual={use_residual} mode={mode} g={g_})")
            assert ratio <= 0.5, f"filter error reaches {ratio:.3f} of the bound E (mode {mode}, group {g_})"
            if K < 256:
                assert (sc[g_][:, K:] < -1e37).all()
            a, _, _ = o.assign(rows[g_], s_np[g_, 0], g_np[g_, 0] if mode == 0 else None)
            assert np.array_equal(idx[g_].cpu().numpy(), a)
