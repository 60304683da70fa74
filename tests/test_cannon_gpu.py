"""NEXT-3 on one GPU: the blocked contraction kernel (foldcp_trimul_contract_blocks -- accumulator
resident in tensor memory across a rank's block pairs) emulating every rank of a g x g mesh in turn
over all ranks' blocks.  (With fewer GPUs than ranks the ranks are run one after another on their own
block pointers; nothing waits on another launch.)  Peer-mapped pointers over NVLink need the
multi-GPU node and are unmeasured here -- DESIGN.md section 8."""
import numpy as np
import pytest
import torch

import parity_util as U
from oracle import trimul_oracle as orc
from paper_2603_14806_b200 import binding as B
from paper_2603_14806_b200 import cannon

pytestmark = pytest.mark.gpu
DEV = "cuda"
OUT, INC = B.OUTGOING, B.INCOMING


def run_grid(a, b, direction, g):
    """o assembled from g*g per-rank calls, each contracting that rank's g block pairs in Cannon order."""
    blocks_a = {k: v.to(DEV) for k, v in cannon.split_blocks(a, g).items()}
    blocks_b = {k: v.to(DEV) for k, v in cannon.split_blocks(b, g).items()}
    N = a.shape[1]
    nb = N // g
    o = None
    for r in range(g):
        for c in range(g):
            steps = cannon.blocks_for_rank(r, c, g, direction)
            ob = B.contract_blocks([blocks_a[s[0]] for s in steps], [blocks_b[s[1]] for s in steps], direction)
            if o is None:
                o = torch.empty(a.shape[0], N, N, dtype=ob.dtype, device=DEV)
            o[:, r * nb:(r + 1) * nb, c * nb:(c + 1) * nb] = ob
    torch.cuda.synchronize()
    return o


@pytest.mark.parametrize("direction", [OUT, INC])
@pytest.mark.parametrize("g,N,dtype", [(2, 528, torch.bfloat16), (2, 512, torch.float16), (4, 1088, torch.bfloat16),
                                       (3, 201, torch.float32), (2, 80, torch.bfloat16)])
def test_blocked_contraction_matches_oracle_cannon(direction, g, N, dtype):
    gen = torch.Generator().manual_seed(17 * g + N)
    a = torch.randn(128, N, N, generator=gen).to(dtype)
    b = torch.randn(128, N, N, generator=gen).to(dtype)
    o = run_grid(a, b, direction, g)
    t = lambda x: np.transpose(U.np64(x), (1, 2, 0))
    ref = orc.contraction_cannon(t(a), t(b), direction, g)
    got = t(o)
    if dtype == torch.float32:
        assert U.errors(got, ref)["rel_fro"] < 1e-5
    else:
        # only the final bf16 rounding of o (2^-9 relative) plus fp32 accumulation
        assert np.abs(got - ref).max() <= 2.0 ** -8 * np.abs(ref).max()
        assert U.errors(got, ref)["rel_fro"] < 3e-3


@pytest.mark.parametrize("direction", [OUT, INC])
def test_blocked_contraction_in_natural_order_is_bitwise_the_monolithic_kernel(direction):
    """Block pairs passed in natural order q = 0, 1 walk k in the same order as one launch over the
    whole tensors, into the same TMEM accumulator: bit-identical output blocks."""
    g, N = 2, 512
    gen = torch.Generator().manual_seed(5)
    a = torch.randn(128, N, N, generator=gen).to(torch.bfloat16)
    b = torch.randn(128, N, N, generator=gen).to(torch.bfloat16)
    whole = B.contract(a.to(DEV), b.to(DEV), direction)
    blocks_a = {k: v.to(DEV) for k, v in cannon.split_blocks(a, g).items()}
    blocks_b = {k: v.to(DEV) for k, v in cannon.split_blocks(b, g).items()}
    nb = N // g
    for r in range(g):
        for c in range(g):
            if direction == OUT:
                la, lb = [blocks_a[(r, q)] for q in range(g)], [blocks_b[(c, q)] for q in range(g)]
            else:
                la, lb = [blocks_a[(q, r)] for q in range(g)], [blocks_b[(q, c)] for q in range(g)]
            ob = B.contract_blocks(la, lb, direction)
            torch.cuda.synchronize()
            assert torch.equal(ob, whole[:, r * nb:(r + 1) * nb, c * nb:(c + 1) * nb])


def test_blocked_contraction_rejects_bad_arguments():
    a = torch.zeros(128, 64, 64, dtype=torch.bfloat16, device=DEV)
    with pytest.raises(B.FoldcpError) as ei:
        B.contract_blocks([a] * 5, [a] * 5, OUT)
    assert ei.value.status == 2
    with pytest.raises(B.FoldcpError) as ei:
        B.contract_blocks([a], [a], OUT, o_block=a)
    assert ei.value.status == 5
