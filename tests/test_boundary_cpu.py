"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol the header
declares, sizes workspaces, and rejects bad arguments before touching CUDA."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def B():
    import __graft_entry__ as ge
    ge.build()
    from paper_2607_01065_b200 import binding
    return binding


def test_every_declared_symbol_is_exported(B):
    hdr = (ROOT / "include" / "gsrq.h").read_text()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(gsrq_[a-z_0-9]+)\s*\(", hdr))
    assert {"gsrq_fit_stage", "gsrq_encode", "gsrq_decode", "gsrq_workspace_bytes"} <= names
    lib = B.lib()
    for n in names:
        assert hasattr(lib, n), n
    assert set(B.EXPORTS) == names
    assert "sm_100a" in B.gsrq_version()


def test_struct_layout_matches_header(B):
    assert C.sizeof(B.gsrq_view) == 40
    assert C.sizeof(B.gsrq_codebook) == 24
    assert C.sizeof(B.gsrq_fit_stats) == 24 + 8 * 128 + 8 * 128


def test_workspace_bytes_and_argument_errors(B):
    v = B.gsrq_view(B.GSRQ_BF16, 8, 4096, 128, 16, 4096 * 128, 128)
    n_all = B.gsrq_workspace_bytes(v, 256, 2, 0)
    n_fit = B.gsrq_workspace_bytes(v, 256, 2, 512)
    assert n_all > n_fit > 8 * 4096 * 8 * 4      # the flagged-row list alone
    assert n_all % 256 == 0
    for bad in [B.gsrq_view(B.GSRQ_BF16, 8, 4096, 128, 24, 4096 * 128, 128),    # hd % d
                B.gsrq_view(7, 8, 4096, 128, 16, 4096 * 128, 128),              # dtype
                B.gsrq_view(B.GSRQ_BF16, 8, 4096, 128, 16, 4096 * 128 + 1, 128)]:  # alignment
        with pytest.raises(B.GsrqError) as e:
            B.gsrq_workspace_bytes(bad, 256, 2, 0)
        assert e.value.code == -1
    with pytest.raises(B.GsrqError):
        B.gsrq_workspace_bytes(v, 257, 2, 0)
    lib = B.lib()
    v4 = B.gsrq_view(B.GSRQ_BF16, 8, 4096, 128, 4, 4096 * 128, 128)      # d = 4: no kernel (GSRQ_EUNSUPPORTED)
    assert lib.gsrq_workspace_bytes(C.byref(v4), 256, 2, C.c_int64(0)) == 0
    assert b"d = 4" in lib.gsrq_last_error()
    for d_wide in (64, 128):                                             # the paper's operating points are served
        vw = B.gsrq_view(B.GSRQ_BF16, 8, 4096, 128, d_wide, 4096 * 128, 128)
        assert lib.gsrq_workspace_bytes(C.byref(vw), 256, 12, C.c_int64(0)) > 0
    # stand-alone clustering (KM baseline / GSKM): argument checks
    assert B.lib().gsrq_cluster_workspace_bytes(C.c_int64(10000), 256, 2048) > 0
    assert B.lib().gsrq_cluster_workspace_bytes(C.c_int64(10000), 258, 2048) == 0     # d not a multiple of 4
    assert B.lib().gsrq_cluster_workspace_bytes(C.c_int64(10000), 256, 5000) == 0     # K > 4096
    # compute entry points validate before any CUDA call: NULL pointers -> GSRQ_EINVAL
    cb = B.gsrq_codebook(256, 2, None, None)
    rc = lib.gsrq_encode(None, C.byref(v), C.byref(cb), 0, 2, None, None, None, C.c_size_t(0), None)
    assert rc == -1
    rc = lib.gsrq_decode(None, C.byref(cb), 2, None, C.byref(v), None)
    assert rc == -1
    # argument checks that come before any CUDA call (fake, never dereferenced addresses)
    p = lambda a: C.c_void_p(a)
    assert lib.gsrq_pack_nibbles(p(0x1000), 17, C.c_int64(1), C.c_int64(8), p(0x2000), None) == -1 and b"K = 17" in lib.gsrq_last_error()
    cb_ok = B.gsrq_codebook(256, 2, 0x10000, 0x20000)
    cb_odd = B.gsrq_codebook(256, 2, 0x10004, 0x20000)   # shapes are read as float4
    attn = lambda fn, kcb, Bq, tail: fn(p(0x1000), p(0x2000), C.byref(kcb), 2, p(0x3000), C.byref(cb_ok), 2, C.c_int64(8 * 64), p(0x4000), p(0x5000),
                                         C.c_int64(64), Bq, 32, 8, 128, 16, C.c_float(0.1), C.c_float(0.0), p(0x6000), *tail)
    ws = (p(0x7000), C.c_size_t(1 << 30), None)
    assert attn(lib.gsrq_attention_decode, cb_odd, 2, ws) == -1 and b"16-byte" in lib.gsrq_last_error()
    assert attn(lib.gsrq_attention_decode, cb_ok, 70000, ws) == -1 and b"65535" in lib.gsrq_last_error()
    assert attn(lib.gsrq_attention_decode_static, cb_odd, 2, (None,)) == -1
    assert attn(lib.gsrq_attention_decode_static, cb_ok, 70000, (None,)) == -1
    assert lib.gsrq_cluster_assign(p(0x1004), C.c_int64(100), 16, 8, 0, p(0x2000), p(0x3000), p(0x4000), None) == -1


def test_product_path_does_not_reach_the_oracle():
    """The CUDA path and its binding must not import or link anything under oracle/."""
    for p in (ROOT / "paper_2607_01065_b200").rglob("*"):
        if p.suffix in {".py", ".cu", ".cuh", ".h"}:
            txt = p.read_text()
            assert not re.search(r"(import\s+oracle|from\s+oracle|#include[^\n]*oracle|gsrq_oracle|oracle/build)", txt), p
