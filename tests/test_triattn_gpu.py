"""Triangle attention: the CUDA path (include/foldcp_triattn.h) against the fp64
oracle (oracle/triattn_oracle.py) on the same seeded inputs, element by element."""
import numpy as np
import pytest
import torch

import parity_util as U
from oracle import triattn_oracle as ta
from paper_2603_14806_b200 import binding as B
from paper_2603_14806_b200 import synth

pytestmark = pytest.mark.gpu
DEV = "cuda"
H, CH, CZ = 4, 32, 128


def make(N, seed, dtype, mask_kind):
    """BASELINE-style init (z ~ N(0,1), weights ~ N(0, 1/fan_in), gamma = 1 + 0.1 N, beta = 0.1 N), rounded
    to bf16 once for the bf16 mode so that both sides see the same values."""
    g = torch.Generator().manual_seed(seed)
    rn = lambda *s: torch.randn(*s, generator=g)
    td = torch.float32 if dtype == "f32" else torch.bfloat16
    z = rn(N, N, CZ).to(td)
    p = dict(ln_gamma=1 + 0.1 * rn(CZ), ln_beta=0.1 * rn(CZ))
    for name, rows in (("w_q", H * CH), ("w_k", H * CH), ("w_v", H * CH), ("w_g", H * CH), ("w_t", H)):
        p[name] = (rn(rows, CZ) / CZ ** 0.5).to(td)
    p["w_o"] = (rn(CZ, H * CH) / (H * CH) ** 0.5).to(td)
    M = None
    if mask_kind != "none":
        m = synth.make_token_mask(mask_kind, N, seed)
        M = synth.pair_mask(m, dtype, "cpu")
        M[:, 0] = 1.0                                     # every line keeps one unmasked key (a fully
        M[0, :] = 1.0                                     # masked softmax row is degenerate: -1e9 + s)
    return z, M, p


def run(N, node, dtype, mask_kind, seed=5):
    z, M, p = make(N, seed, dtype, mask_kind)
    out = B.triattn(z.to(DEV), None if M is None else M.to(DEV), {k: v.to(DEV) for k, v in p.items()}, node)
    torch.cuda.synchronize()
    ref = ta.triangle_attention(U.np64(z), None if M is None else U.np64(M),
                                {k: U.np64(v) for k, v in p.items()}, node, H)
    e = U.errors(U.np64(out), ref)
    U.record_parity(f"triattn {dtype} N={N} node={node} mask={mask_kind}", e, "f32" if dtype == "f32" else "bf16", N=N)
    return e


@pytest.mark.parametrize("node", [B.TRIATTN_STARTING, B.TRIATTN_ENDING])
@pytest.mark.parametrize("N,mask_kind", [(1, "none"), (5, "none"), (67, "tail"), (130, "scatter"), (264, "tail")])
def test_triattn_fp32(node, N, mask_kind):
    e = run(N, node, "f32", mask_kind)
    assert e["rel_fro"] <= 1e-5 and e["max_over_rms"] <= 1e-4, e


@pytest.mark.parametrize("node", [B.TRIATTN_STARTING, B.TRIATTN_ENDING])
@pytest.mark.parametrize("N,mask_kind", [(8, "none"), (136, "scatter"), (264, "tail"), (512, "tail")])
def test_triattn_bf16(node, N, mask_kind):
    # bf16 storage of z / weights / out, fp32 arithmetic: only the output rounding (2^-9) remains
    e = run(N, node, "bf16", mask_kind)
    assert e["rel_fro"] <= 3e-3 and e["max_over_rms"] <= 5e-2, e


def test_triattn_nodes_differ_and_are_deterministic():
    z, M, p = make(72, 3, "bf16", "tail")
    zd, Md, pd = z.to(DEV), M.to(DEV), {k: v.to(DEV) for k, v in p.items()}
    a = B.triattn(zd, Md, pd, B.TRIATTN_STARTING)
    b = B.triattn(zd, Md, pd, B.TRIATTN_ENDING)
    a2 = B.triattn(zd, Md, pd, B.TRIATTN_STARTING)
    torch.cuda.synchronize()
    assert torch.equal(a, a2) and not torch.equal(a, b)
    # ending node == starting node on the transposed input (exactly the same arithmetic per output)
    c = B.triattn(zd.transpose(0, 1).contiguous(), Md.t().contiguous(), pd, B.TRIATTN_STARTING)
    torch.cuda.synchronize()
    assert torch.equal(b, c.transpose(0, 1).contiguous())


def test_triattn_rejects_bad_arguments():
    z, M, p = make(16, 1, "bf16", "none")
    zd, pd = z.to(DEV), {k: v.to(DEV) for k, v in p.items()}
    with pytest.raises(B.FoldcpError) as ei:
        B.triattn(zd, None, pd, 2)
    assert ei.value.status == 1
    with pytest.raises(B.FoldcpError) as ei:
        B.triattn(zd, None, pd, 0, workspace=torch.empty(256, dtype=torch.uint8, device=DEV))
    assert ei.value.status == 4
    with pytest.raises(B.FoldcpError) as ei:
        B.triattn(zd, None, pd, 0, out=zd)
    assert ei.value.status == 5
    assert B.triattn_workspace_bytes(16, 64) == 0 and B.triattn_workspace_bytes(16, 128, 8) == 0
    # bf16 mode needs N % 8 == 0 (16-byte TMA strides); the fp32 mode takes any N
    assert B.triattn_workspace_bytes(12, dtype=B.BF16) == 0 and B.triattn_workspace_bytes(12, dtype=B.F32) > 0
    z12 = torch.zeros(12, 12, 128, dtype=torch.bfloat16, device=DEV)
    with pytest.raises(B.FoldcpError) as ei:
        B.triattn(z12, None, pd, 0)
    assert ei.value.status == 2
