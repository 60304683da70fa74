"""foldcp_trimul_static: the entry point that allocates nothing (scratch in a static __device__ array
of the library, include/foldcp_trimul.h).  Checked against the existing path (foldcp_trimul with a
caller-owned workspace: same kernels, so bitwise) and against the oracle within the parity
tolerance, on two calls in a row that share the array.

Collected LAST on purpose (file name): the run uses `pytest -x`."""
import pytest
import torch

import parity_util as U
from paper_2603_14806_b200 import binding as B
from paper_2603_14806_b200 import synth

DEV = "cuda"
OUT, INC = B.OUTGOING, B.INCOMING
STATIC_LIMIT = 8     # FOLDCP_ERR_STATIC_LIMIT


def _dev(p):
    return {k: v.to(DEV) for k, v in p.items()}


def test_static_limits_match_workspace_bytes():
    """host logic only: the stated maximum is the workspace formula against 16 MiB"""
    cap = B.static_workspace_bytes()
    assert cap == 16 << 20
    for dt, step, expect in ((B.BF16, 8, 144), (B.F32, 1, 104)):
        n = B.static_max_n(dt)
        assert n == expect
        assert B.workspace_bytes(n, 128, 128, dt) <= cap < B.workspace_bytes(n + step, 128, 128, dt)
    assert B.static_max_n(B.BF16, c_z=64) == 0      # unsupported shape
    assert "static workspace" in B.status_string(STATIC_LIMIT)


@pytest.mark.gpu
@pytest.mark.parametrize("cfg_index,sizes", [(1, (136, 72)), (0, (67, 104))])
def test_static_matches_existing_path_two_calls_in_a_row(cfg_index, sizes):
    """Call 1 and call 2 differ in N, direction, inputs and mask, so anything call 1 leaves in the
    shared array (a, b, o, statistics, tile counters) would show in call 2."""
    cfg = synth.CONFIGS[cfg_index]
    cases = []
    for N, direction, kind in ((sizes[0], OUT, "scatter"), (sizes[1], INC, "tail")):
        z, M, p = synth.make_inputs(cfg, direction, "cpu", N=N)
        M = synth.pair_mask(synth.make_token_mask(kind, N, cfg.seed + N), cfg.dtype)
        cases.append((z, M, p, direction))
    dev = [(z.to(DEV), M.to(DEV), _dev(p), torch.empty_like(z, device=DEV)) for z, M, p, _ in cases]
    # the existing path first (it also loads the kernels, so the memory reading below is steady)
    want = [B.trimul(zd, Md, pd, c[3]) for (zd, Md, pd, _), c in zip(dev, cases)]
    torch.cuda.synchronize()

    got = [B.trimul_static(zd, Md, pd, c[3], out) for (zd, Md, pd, out), c in zip(dev, cases)]
    torch.cuda.synchronize()
    for i, ((z, M, p, direction), w, g) in enumerate(zip(cases, want, got)):
        assert torch.equal(g, w), f"call {i + 1}: static path differs from the workspace path"
        ref = U.oracle_full(z, M, p, direction)
        U.assert_parity(U.np64(g), ref, cfg.dtype, f"static call {i + 1} cfg{cfg.index} N={z.shape[0]}")

    # once more in the opposite order (call 1's problem after call 2's leftovers), watching the
    # device memory: the first call above loaded the module that holds the 16 MiB array (the array
    # itself, resident from then on); from here on nothing may be allocated, by torch or the library
    for i in (1, 0):
        dev[i][3].zero_()
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    torch_bytes0 = torch.cuda.memory_allocated()
    for i in (1, 0):
        zd, Md, pd, out = dev[i]
        B.trimul_static(zd, Md, pd, cases[i][3], out)
    torch.cuda.synchronize()
    # (<=: Python may collect earlier tests' tensors in between)
    assert torch.cuda.memory_allocated() <= torch_bytes0
    free1, _ = torch.cuda.mem_get_info()
    # an allocated workspace would be 3.6 - 16 MB
    assert free0 - free1 < (2 << 20), f"device memory dropped by {free0 - free1} bytes"
    for i in (1, 0):
        assert torch.equal(dev[i][3], want[i])


@pytest.mark.gpu
def test_static_rejects_sizes_beyond_the_maximum():
    for cfg_index, N in ((1, 152), (0, 105)):
        cfg = synth.CONFIGS[cfg_index]
        z, M, p = synth.make_inputs(cfg, OUT, "cpu", N=N)
        out = torch.full_like(z, 7.0, device=DEV)
        with pytest.raises(B.FoldcpError) as e:
            B.trimul_static(z.to(DEV), M.to(DEV), _dev(p), OUT, out)
        assert e.value.status == STATIC_LIMIT
        torch.cuda.synchronize()
        assert bool((out == 7.0).all())          # nothing was launched
    # the largest accepted size runs
    cfg = synth.CONFIGS[1]
    N = B.static_max_n(B.BF16)
    z, M, p = synth.make_inputs(cfg, INC, "cpu", N=N)
    zd, Md, pd = z.to(DEV), M.to(DEV), _dev(p)
    got = B.trimul_static(zd, Md, pd, INC, torch.empty_like(zd))
    want = B.trimul(zd, Md, pd, INC)
    torch.cuda.synchronize()
    assert torch.equal(got, want)
