"""NEXT-3 host logic on the CPU: the block bookkeeping of the Cannon-style distributed contraction
(paper_2603_14806_b200/cannon.py) against the oracle's simulated grid, and a world_size-4 gloo run in
which four processes really exchange blocks by P2P following `ring_plan` (transpose, alignment, g ring
steps) and reproduce the serial contraction."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import trimul_oracle as orc
from paper_2603_14806_b200 import cannon

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("g", [1, 2, 3, 4])
@pytest.mark.parametrize("direction", [0, 1])
def test_blocks_for_rank_matches_oracle_schedule(g, direction):
    sched = orc.cannon_schedule(g, direction)
    for r in range(g):
        for c in range(g):
            assert cannon.blocks_for_rank(r, c, g, direction) == sched[(r, c)]


def test_grid_side_requires_a_square():
    assert cannon.grid_side(4) == 2 and cannon.grid_side(16) == 4 and cannon.grid_side(1) == 1
    with pytest.raises(ValueError):
        cannon.grid_side(8)


def _exchange(send_t, dst, recv_like, src, rank):
    """deadlock-free P2P exchange (self-sends are copies)"""
    if dst == rank and src == rank:
        return send_t.clone()
    out = torch.empty_like(recv_like)
    reqs = [dist.isend(send_t.contiguous(), dst), dist.irecv(out, src)]
    for q in reqs:
        q.wait()
    return out


def _worker(rank, world, port, direction, N, c, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        g = cannon.grid_side(world)
        r, cc = cannon.rank_to_coord(rank, g)
        gen = torch.Generator().manual_seed(123)
        a = torch.randn(c, N, N, generator=gen, dtype=torch.float64)
        b = torch.randn(c, N, N, generator=gen, dtype=torch.float64)
        my_a = cannon.split_blocks(a, g)[(r, cc)]
        my_b = cannon.split_blocks(b, g)[(r, cc)]
        plan = cannon.ring_plan(r, cc, g, direction)
        # 1. transpose one operand across the grid
        if plan["transposed_operand"] == "b":
            my_b = _exchange(my_b, plan["transpose_peer"], my_b, plan["transpose_peer"], rank)
        else:
            my_a = _exchange(my_a, plan["transpose_peer"], my_a, plan["transpose_peer"], rank)
        # 2. Cannon's initial alignment
        my_a = _exchange(my_a, plan["align_a_to"], my_a, plan["align_a_from"], rank)
        my_b = _exchange(my_b, plan["align_b_to"], my_b, plan["align_b_from"], rank)
        want = cannon.blocks_for_rank(r, cc, g, direction)
        blocks_a, blocks_b = cannon.split_blocks(a, g), cannon.split_blocks(b, g)
        nb = N // g
        acc = np.zeros((nb, nb, c))
        for s in range(g):
            # the resident blocks are exactly the ones the schedule names for this step
            assert torch.equal(my_a, blocks_a[want[s][0]]) and torch.equal(my_b, blocks_b[want[s][1]])
            acc += orc.contraction(my_a.permute(1, 2, 0).numpy(), my_b.permute(1, 2, 0).numpy(), direction)
            if s + 1 < g:
                my_a = _exchange(my_a, plan["shift_a_to"], my_a, plan["shift_a_from"], rank)
                my_b = _exchange(my_b, plan["shift_b_to"], my_b, plan["shift_b_from"], rank)
        full = orc.contraction(a.permute(1, 2, 0).numpy(), b.permute(1, 2, 0).numpy(), direction)
        ref = full[r * nb:(r + 1) * nb, cc * nb:(cc + 1) * nb]
        err = float(np.abs(acc - ref).max() / np.abs(ref).max())
        gathered = [None] * world
        dist.all_gather_object(gathered, err)
        if rank == 0:
            ret.put(gathered)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("direction", [0, 1])
def test_world_size_4_gloo_ring_reproduces_the_serial_contraction(direction):
    world, port = 4, 29613 + direction
    ctx = mp.get_context("spawn")
    ret = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(rk, world, port, direction, 8, 3, ret)) for rk in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    errs = ret.get(timeout=10)
    assert len(errs) == 4 and max(errs) < 1e-13
