"""Block bookkeeping of the paper's Cannon-style distributed triangle multiplication
(Fig. 2b, Table 1 line 83).

The pair tensors are tiled as (N / g)^2 blocks on a g x g mesh (g = sqrt(P), the paper's square
topology, lines 77-79); rank (r, c) owns block (r, c) of a and of b.  In ring step s it multiplies
the two blocks whose contracted block index is q = (r + c + s) mod g:

    outgoing  o_(r,c) += a_(r,q) b_(c,q)^T        incoming  o_(r,c) += a_(q,r)^T b_(q,c)

This module holds index arithmetic only (which rank owns / sends / receives which block when);
the arithmetic runs in the library: `binding.contract_blocks` contracts a rank's block pairs in ONE
kernel whose accumulator stays in tensor memory.  On an NVLink / NVSwitch node every peer is one hop
away, so the block pointers of the other ranks can be peer-mapped and read directly by that kernel's
TMA loads (no store-and-forward ring); `ring_plan` gives the paper's explicit send / receive
schedule for a transport that wants it (and for the CPU test with gloo).
"""
from __future__ import annotations

from typing import Dict, List, Tuple

OUTGOING = 0
INCOMING = 1
Block = Tuple[int, int]


def grid_side(world_size: int) -> int:
    """sqrt(P); the CP world size must be a perfect square."""
    g = int(round(world_size ** 0.5))
    if g * g != world_size:
        raise ValueError(f"context-parallel world size {world_size} is not a perfect square")
    return g


def rank_to_coord(rank: int, g: int) -> Block:
    return rank // g, rank % g


def coord_to_rank(r: int, c: int, g: int) -> int:
    return (r % g) * g + (c % g)


def blocks_for_rank(r: int, c: int, g: int, direction: int) -> List[Tuple[Block, Block]]:
    """[(a block, b block) for ring step s = 0 .. g-1] that rank (r, c) multiplies, Cannon order."""
    steps = []
    for s in range(g):
        q = (r + c + s) % g
        steps.append((((r, q), (c, q)) if direction == OUTGOING else ((q, r), (q, c))))
    return steps


def ring_plan(r: int, c: int, g: int, direction: int) -> Dict[str, object]:
    """The explicit data movement of the paper's algorithm for rank (r, c):

      transpose: the operand that is transposed across the grid ("b" outgoing, "a" incoming) goes
                 to / comes from rank (c, r);
      align:     Cannon's initial alignment -- a from (r, c + r), b from (r + c, c);
      shift:     every step a is received from the right neighbour (r, c + 1) and sent to the left
                 one (r, c - 1); b is received from below (r + 1, c) and sent up (r - 1, c).
    All entries are ranks (row-major r * g + c)."""
    return {
        "transposed_operand": "b" if direction == OUTGOING else "a",
        "transpose_peer": coord_to_rank(c, r, g),
        "align_a_from": coord_to_rank(r, c + r, g), "align_a_to": coord_to_rank(r, c - r, g),
        "align_b_from": coord_to_rank(r + c, c, g), "align_b_to": coord_to_rank(r - c, c, g),
        "shift_a_from": coord_to_rank(r, c + 1, g), "shift_a_to": coord_to_rank(r, c - 1, g),
        "shift_b_from": coord_to_rank(r + 1, c, g), "shift_b_to": coord_to_rank(r - 1, c, g),
    }


def split_blocks(t, g: int):
    """[c, N, N] channel-major tensor -> {(r, c): contiguous [c, N/g, N/g] block} (torch or numpy)."""
    N = t.shape[1]
    if N % g != 0:
        raise ValueError("N must be divisible by the grid side")
    nb = N // g
    out = {}
    for r in range(g):
        for c in range(g):
            blk = t[:, r * nb:(r + 1) * nb, c * nb:(c + 1) * nb]
            out[(r, c)] = blk.contiguous() if hasattr(blk, "contiguous") else blk.copy()
    return out
