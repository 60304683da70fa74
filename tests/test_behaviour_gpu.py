"""GPU behaviour tests through the C ABI: determinism, mask / bias conventions, invariants that hold
at any size (I1, I2, I3), streams, workspace bounds, error codes on a live device."""
import ctypes
import threading

import numpy as np
import pytest
import torch

import parity_util as U
from paper_2603_14806_b200 import binding as B
from paper_2603_14806_b200 import synth

pytestmark = pytest.mark.gpu
DEV = "cuda"
OUT, INC = B.OUTGOING, B.INCOMING


def inputs(N, direction=OUT, cfg_idx=1, mask_kind="tail"):
    cfg = synth.CONFIGS[cfg_idx]
    z, _, p = synth.make_inputs(cfg, direction, "cpu", N=N)
    M = synth.pair_mask(synth.make_token_mask(mask_kind, N, cfg.seed), cfg.dtype)
    return z.to(DEV), M.to(DEV), {k: v.to(DEV) for k, v in p.items()}


@pytest.mark.parametrize("direction", [OUT, INC])
def test_bitwise_deterministic(direction):
    z, M, p = inputs(520, direction)
    o1 = B.trimul(z, M, p, direction)
    o2 = B.trimul(z, M, p, direction)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2)


def test_null_mask_equals_ones_mask():
    z, M, p = inputs(136)
    o1 = B.trimul(z, None, p, OUT)
    o2 = B.trimul(z, torch.ones_like(M), p, OUT)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2)


def test_null_biases_equal_zero_biases_and_match_oracle():
    z, M, p = inputs(72)
    q = dict(p)
    pz = dict(p)
    for k in ("b_a", "b_a_gate", "b_b", "b_b_gate", "b_g", "b_o"):
        q[k] = None
        pz[k] = torch.zeros_like(p[k])
    o1 = B.trimul(z, M, q, INC)
    o2 = B.trimul(z, M, pz, INC)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2)
    ref = U.oracle_full(z, M, {k: v for k, v in q.items() if v is not None}, INC)
    U.assert_parity(U.np64(o1), ref, "bf16", "no-bias")


@pytest.mark.parametrize("direction", [OUT, INC])
def test_I3_garbage_under_mask_is_bitwise_invisible(direction):
    z, M, p = inputs(264, direction, mask_kind="scatter")
    z2 = z.clone()
    dead = (M == 0)
    z2[dead] = (100.0 * torch.randn(int(dead.sum()), 128, device=DEV)).to(z.dtype)
    o1 = B.trimul(z, M, p, direction)
    o2 = B.trimul(z2, M, p, direction)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2)
    assert torch.all(o1[dead] == 0)
    # without the output mask: valid pairs still bitwise equal, masked pairs non-zero (A8 / A20)
    n1 = B.trimul(z, M, p, direction, mask_output=False)
    n2 = B.trimul(z2, M, p, direction, mask_output=False)
    torch.cuda.synchronize()
    assert torch.equal(n1[~dead], n2[~dead])
    assert torch.equal(n1[~dead], o1[~dead])
    assert n1[dead].float().abs().max() > 0


def test_I1_direction_identity_with_ab_swap():
    z, M, p = inputs(200, INC)
    sw = dict(p)
    for x, y in (("w_a", "w_b"), ("w_a_gate", "w_b_gate"), ("b_a", "b_b"), ("b_a_gate", "b_b_gate")):
        sw[x], sw[y] = p[y], p[x]
    inc = B.trimul(z, M, p, INC)
    out = B.trimul(z.transpose(0, 1).contiguous(), M.t().contiguous(), sw, OUT).transpose(0, 1)
    torch.cuda.synchronize()
    e = U.errors(U.np64(out), U.np64(inc))
    assert e["rel_fro"] < 2e-2 and e["max_over_rms"] < 1e-1      # 2x the parity tolerance


def test_I2_token_permutation_equivariance():
    z, M, p = inputs(200, OUT, mask_kind="scatter")
    pi = torch.randperm(200, generator=torch.Generator().manual_seed(3)).to(DEV)
    lhs = B.trimul(z[pi][:, pi].contiguous(), M[pi][:, pi].contiguous(), p, OUT)
    rhs = B.trimul(z, M, p, OUT)[pi][:, pi]
    torch.cuda.synchronize()
    e = U.errors(U.np64(lhs), U.np64(rhs))
    assert e["rel_fro"] < 2e-2 and e["max_over_rms"] < 1e-1


def test_non_default_stream_is_asynchronous_and_correct():
    z, M, p = inputs(264)
    ref = B.trimul(z, M, p, OUT)
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        got = B.trimul(z, M, p, OUT)
        ev = torch.cuda.Event()
        ev.record(s)
    ev.synchronize()
    assert torch.equal(got, ref)


def test_two_host_threads_two_streams():
    z, M, p = inputs(136)
    ref = B.trimul(z, M, p, OUT)
    torch.cuda.synchronize()
    res = [None, None]

    def work(i):
        torch.cuda.set_device(0)
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            for _ in range(5):
                res[i] = B.trimul(z, M, p, OUT)
        s.synchronize()

    ts = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    [t.start() for t in ts]
    [t.join() for t in ts]
    assert torch.equal(res[0], ref) and torch.equal(res[1], ref)


def test_workspace_bound_is_respected():
    N = 136
    z, M, p = inputs(N)
    need = B.workspace_bytes(N)
    ws = torch.full((need + 4096,), 0x5A, dtype=torch.uint8, device=DEV)
    B.trimul(z, M, p, OUT, workspace=ws[:need])
    torch.cuda.synchronize()
    assert torch.all(ws[need:] == 0x5A)
    with pytest.raises(B.FoldcpError) as ei:
        B.trimul(z, M, p, OUT, workspace=ws[:need - 256])
    assert ei.value.status == 4


def test_error_codes_leave_out_untouched():
    z, M, p = inputs(72)
    out = torch.full_like(z, 7.0)
    with pytest.raises(B.FoldcpError) as ei:
        B.trimul(z, M, p, 2, out=out)
    assert ei.value.status == 1
    with pytest.raises(B.FoldcpError) as ei:
        B.trimul(z, M, p, OUT, out=z)
    assert ei.value.status == 5
    torch.cuda.synchronize()
    assert torch.all(out == 7.0)
