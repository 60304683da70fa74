"""C-ABI checks that need no GPU: the library builds/loads, exports every symbol the header
declares, and rejects bad arguments on the host before touching the device."""
import ctypes
import os
import re

import pytest

from paper_2603_14806_b200 import binding as B
from paper_2603_14806_b200 import build as builder

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    builder.build()
    return B.load()


def test_exports_match_header(lib):
    # every entry point declared in include/*.h is exported by the library and bound, and vice versa
    hdr = "".join(open(os.path.join(ROOT, "include", f)).read()
                  for f in ("foldcp_trimul.h", "foldcp_triattn.h"))
    declared = set(re.findall(r"\b(foldcp_[a-z_]+)\s*\(", hdr))
    assert declared == set(B.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_version_and_strings(lib):
    assert B.version() >= 100
    assert B.status_string(0) == "ok"
    assert "workspace" in B.status_string(4)
    assert B.status_string(99) == "unknown status"


def test_workspace_bytes(lib):
    # a, b, o (12 GiB) + the LayerNorm(z) statistics K1 hands to K3 (8 bytes per pair) + counters
    assert B.workspace_bytes(4096, 128, 128, B.BF16) == 3 * 128 * 4096 * 4096 * 2 + 8 * 4096 * 4096 + 256
    assert B.workspace_bytes(8192, 128, 128, B.BF16) == 48 * 2 ** 30 + 8 * 8192 * 8192 + B.SCHED_SCRATCH_BYTES
    assert B.workspace_bytes(64, 128, 128, B.F32) == 3 * 128 * 64 * 64 * 4 + 256
    assert B.workspace_bytes(12, 128, 128, B.BF16) == 0      # N % 8 != 0 in bf16
    assert B.workspace_bytes(12, 128, 128, B.F32) > 0
    assert B.workspace_bytes(64, 64, 128, B.BF16) == 0       # c_z != 128
    assert B.workspace_bytes(64, 128, 64, B.BF16) == 0
    assert B.workspace_bytes(0, 128, 128, B.BF16) == 0
    assert B.workspace_bytes(64, 128, 128, 7) == 0
    prev = 0
    for n in (8, 64, 512, 2048, 4096, 8192):                 # monotone in N
        cur = B.workspace_bytes(n)
        assert cur > prev
        prev = cur


def _params(lib, dtype=B.BF16, ws=0x10000, ws_bytes=1 << 40):
    s = B._Params()
    s.struct_size = ctypes.sizeof(B._Params)
    s.dtype = dtype
    s.ln_eps = 1e-5
    s.mask_output = 1
    fake = 0x1000    # never dereferenced: all of these calls must fail on the host first
    ptrs = [n for n, t in B._Params._fields_ if t is ctypes.c_void_p and n != "workspace"]
    assert len(ptrs) == 16
    for i, name in enumerate(ptrs):
        setattr(s, name, fake + 0x100 * i)
    s.workspace = ws
    s.workspace_bytes = ws_bytes
    return s


def _call(lib, s, z=0x100000, mask=None, N=64, c_z=128, c=128, direction=0, out=0x900000):
    return lib.foldcp_trimul(z, mask, ctypes.byref(s) if s is not None else None, N, c_z, c,
                             direction, out, None)


def test_host_side_rejections(lib):
    INVALID, UNSUPPORTED, ALIGN, WS, ALIAS = 1, 2, 3, 4, 5
    assert _call(lib, None) == INVALID
    s = _params(lib)
    assert _call(lib, s, z=None) == INVALID
    assert _call(lib, s, out=None) == INVALID
    assert _call(lib, s, N=0) == INVALID
    assert _call(lib, s, N=-4) == INVALID
    assert _call(lib, s, direction=2) == INVALID
    assert _call(lib, s, N=12) == UNSUPPORTED
    assert _call(lib, s, c_z=64) == UNSUPPORTED
    assert _call(lib, s, c=64) == UNSUPPORTED
    assert _call(lib, s, z=0x100002) == ALIGN
    assert _call(lib, s, out=0x900008) == ALIGN
    assert _call(lib, s, mask=0x500004) == ALIGN
    bad = _params(lib); bad.struct_size -= 4
    assert _call(lib, bad) == INVALID
    bad = _params(lib); bad.dtype = 7
    assert _call(lib, bad) == INVALID
    bad = _params(lib); bad.add_residual = 2
    assert _call(lib, bad) == INVALID
    bad = _params(lib); bad.reserved0 = 1
    assert _call(lib, bad) == INVALID
    bad = _params(lib); bad.mask_output = 5
    assert _call(lib, bad) == INVALID
    assert lib.foldcp_trimul_batched(0x100000, None, ctypes.byref(_params(lib)), 0, 64, 128, 128, 0,
                                     0x900000, None) == INVALID
    for name in ("ln_in_gamma", "w_a", "w_b_gate", "w_g", "ln_out_beta", "w_o"):
        bad = _params(lib); setattr(bad, name, None)
        assert _call(lib, bad) == INVALID, name
    bad = _params(lib); bad.w_a = 0x1002
    assert _call(lib, bad) == ALIGN
    need = B.workspace_bytes(64)
    assert _call(lib, _params(lib, ws=None)) == WS
    assert _call(lib, _params(lib, ws_bytes=need - 1)) == WS
    # aliasing: out == z, out inside the workspace, z inside the workspace
    big = 0x40000000
    assert _call(lib, _params(lib, ws=big, ws_bytes=need), z=0x100000, out=0x100000) == ALIAS
    assert _call(lib, _params(lib, ws=big, ws_bytes=need), out=big + 4096) == ALIAS
    assert _call(lib, _params(lib, ws=big, ws_bytes=need), z=big + 256) == ALIAS


def test_stage_entry_points_reject_aliasing_and_missing_scratch(lib):
    """The persistent kernels store tiles while later tiles still read the operands, so an in-place
    stage call must be refused on the host; bf16 stage calls need the tile-counter scratch."""
    WS, ALIGN, ALIAS = 4, 3, 5
    s = _params(lib)
    X, Y, Zp, SC = 0x10000000, 0x20000000, 0x30000000, 0x50000000
    by = ctypes.byref(s)
    assert lib.foldcp_trimul_project(X, None, by, 64, 128, 128, X, Y, SC, None) == ALIAS        # a == z
    assert lib.foldcp_trimul_project(X, None, by, 64, 128, 128, Y, Y + 4096, SC, None) == ALIAS  # a, b overlap
    assert lib.foldcp_trimul_project(X, None, by, 64, 128, 128, Y, Zp, None, None) == WS
    assert lib.foldcp_trimul_project(X, None, by, 64, 128, 128, Y, Zp, SC + 8, None) == ALIGN
    assert lib.foldcp_trimul_contract(X, Y, 64, 128, B.BF16, 0, X, SC, None) == ALIAS           # o == a
    assert lib.foldcp_trimul_contract(X, Y, 64, 128, B.BF16, 1, Y + 256, SC, None) == ALIAS      # o inside b
    assert lib.foldcp_trimul_contract(X, Y, 64, 128, B.BF16, 0, Zp, None, None) == WS
    assert lib.foldcp_trimul_contract_backward(X, Y, Zp, 64, 128, B.BF16, 0, 0x60000000, 0x70000000,
                                               None, None) == WS
    assert lib.foldcp_trimul_finalize(X, Y, None, by, 64, 128, 128, X, None) == ALIAS            # out == o
    assert lib.foldcp_trimul_finalize(X, Y, None, by, 64, 128, 128, Y, None) == ALIAS            # out == z


def test_library_has_no_device_global_state_and_reads_no_environment():
    """no __device__ global scheduler pool, no getenv dispatch in the shipped
    build (the A/B knobs exist only under -DFOLDCP_DEBUG_KNOBS)."""
    csrc = os.path.join(ROOT, "paper_2603_14806_b200", "csrc")
    for name in os.listdir(csrc):
        src = open(os.path.join(csrc, name)).read()
        assert "__device__ unsigned int g_" not in src, name
        for line in src.splitlines():
            if "getenv(" in line:
                assert name == "common.h" and "return getenv(name);" in line, (name, line)
    assert "-DFOLDCP_DEBUG_KNOBS" not in " ".join(builder.NVCC_FLAGS)


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "lib_path", lambda: str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        B.load()
