"""Full backward pass through the C ABI against the fp64
oracle's trimul_backward: d_z and every one of the 16 parameter gradients, element by element."""
import numpy as np
import pytest
import torch

import parity_util as U
from oracle import trimul_oracle as orc
from paper_2603_14806_b200 import binding as B
from paper_2603_14806_b200 import synth

pytestmark = pytest.mark.gpu
DEV = "cuda"
OUT, INC = B.OUTGOING, B.INCOMING


def run_backward(cfg, N, direction, mask_kind, mask_output=True, residual=False, drop_bias=()):
    z, _, p = synth.make_inputs(cfg, direction, "cpu", N=N)
    M = synth.pair_mask(synth.make_token_mask(mask_kind, N, cfg.seed), cfg.dtype)
    p = {k: (None if k in drop_bias else v) for k, v in p.items()}
    g = torch.Generator().manual_seed(4242 + N)
    d_out = torch.randn(z.shape, generator=g).to(z.dtype)
    q = {k: v for k, v in U.params64(p).items() if v is not None}
    ref_dz, ref_g = orc.trimul_backward(U.np64(d_out), U.np64(z), U.np64(M), q, direction,
                                        mask_output=mask_output, residual=residual)
    d_z, grads = B.trimul_backward(d_out.to(DEV), z.to(DEV), M.to(DEV),
                                   {k: (None if v is None else v.to(DEV)) for k, v in p.items()},
                                   direction, mask_output=mask_output, residual=residual)
    torch.cuda.synchronize()
    assert set(grads) == set(ref_g)
    res = {"d_z": U.errors(U.np64(d_z), ref_dz)}
    for k in ref_g:
        res[k] = U.errors(U.np64(grads[k]), ref_g[k])
    return res


@pytest.mark.parametrize("direction", [OUT, INC])
@pytest.mark.parametrize("N", [64, 37])
def test_backward_fp32_config0(direction, N):
    """fp32 exact mode: relative Frobenius <= 1e-5 for d_z and every parameter gradient."""
    res = run_backward(synth.CONFIGS[0], N, direction, "tail" if N == 37 else "ones")
    for k, e in res.items():
        U.record_parity(f"backward fp32 N={N} dir={direction} {k}", e, "f32", N=N)
        assert e["rel_fro"] <= 1e-5, (k, e)


@pytest.mark.parametrize("direction", [OUT, INC])
def test_backward_bf16_config1(direction):
    """bf16 mode at config 1 (N = 512, last 10 % of tokens masked): north_star tolerances on d_z
    (rel-F 1e-2, max 5e-2 rms) and rel-F 1e-2 on every parameter gradient."""
    res = run_backward(synth.CONFIGS[1], 512, direction, "tail")
    for k, e in res.items():
        U.record_parity(f"backward bf16 N=512 dir={direction} {k}", e, "bf16", N=512)
        assert e["rel_fro"] <= 1e-2, (k, e)
    assert res["d_z"]["max_over_rms"] <= 5e-2


@pytest.mark.parametrize("N,direction,mask_output,residual,drop", [
    (136, OUT, False, False, ("b_a", "b_g")),
    (200, INC, True, True, ("b_o", "b_b_gate")),
    (8, OUT, True, False, ()),
])
def test_backward_bf16_variants(N, direction, mask_output, residual, drop):
    res = run_backward(synth.CONFIGS[1], N, direction, "scatter", mask_output=mask_output,
                       residual=residual, drop_bias=drop)
    for k, e in res.items():
        assert e["rel_fro"] <= 1e-2, (k, e)


def test_backward_is_bitwise_deterministic():
    cfg = synth.CONFIGS[1]
    N = 264
    z, _, p = synth.make_inputs(cfg, OUT, "cpu", N=N)
    M = synth.pair_mask(synth.make_token_mask("scatter", N, cfg.seed), cfg.dtype).to(DEV)
    z, p = z.to(DEV), {k: v.to(DEV) for k, v in p.items()}
    d_out = torch.randn(z.shape, device=DEV, generator=torch.Generator(device=DEV).manual_seed(1)).to(z.dtype)
    r1 = B.trimul_backward(d_out, z, M, p, OUT)
    r2 = B.trimul_backward(d_out, z, M, p, OUT)
    torch.cuda.synchronize()
    assert torch.equal(r1[0], r2[0])
    for k in r1[1]:
        assert torch.equal(r1[1][k], r2[1][k]), k


def test_backward_rejects_bad_arguments():
    cfg = synth.CONFIGS[1]
    z, _, p = synth.make_inputs(cfg, OUT, "cpu", N=72)
    z, p = z.to(DEV), {k: v.to(DEV) for k, v in p.items()}
    d_out = torch.ones_like(z)
    with pytest.raises(B.FoldcpError) as ei:
        B.trimul_backward(d_out, z, None, p, OUT, workspace=torch.empty(4096, dtype=torch.uint8, device=DEV))
    assert ei.value.status == 4
    with pytest.raises(B.FoldcpError) as ei:
        B.trimul_backward(d_out, z, None, p, 3)
    assert ei.value.status == 1
