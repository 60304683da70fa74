"""fp64 CPU oracle of the triangle multiplicative update (outgoing / incoming).

TEST INFRASTRUCTURE -- NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / `--impl reference` legs may import this package.  It shares no
code with the CUDA path (paper_2603_14806_b200/csrc) and never imports it.

What it computes (plain definition, written out; numpy fp64 throughout):

  PAPER.md lines 117-130, section 3.3, Eq. 2-3 (Eq. 2 is printed twice -- extraction
  duplicate):
      outgoing:  o_nm = sum_k a_nk (.) b_mk          incoming:  o_nm = sum_k a_kn (.) b_km
  "where a, b are projections of the pair representation z in R^{B x N x N x D}.  This
  operation is structurally a batched matrix multiplication with element-wise gating";
  PAPER.md line 132: "The outgoing and incoming variants differ only in which operand is
  transposed".  The paper's equations leave out the LayerNorms, the gates and the output
  projection; BASELINE.json's north_star (= AF3 supplementary Alg. 12/13) fixes them:

      z'   = LayerNorm(z)                                  (over c_z, biased variance)
      a    = M * sigmoid(W_ga z' + b_ga) * (W_a z' + b_a)   (pair mask M applied)
      b    = M * sigmoid(W_gb z' + b_gb) * (W_b z' + b_b)
      g    = sigmoid(W_g z' + b_g)
      o    = contraction above (per channel, no residual add: DESIGN.md reading A1)
      out  = [M *] g * (W_o LayerNorm(o) + b_o)             (LayerNorm over c_hidden)

Readings of the paper taken here are listed in DESIGN.md ("Readings"): A1 update only (no
`+=` residual), A6 eps inside the sqrt / biased variance, A7 pair mask multiplied after
gating, A8 `mask_output` flag.

A library primitive (numpy matmul) serves as the dense-contraction step; there is no
blocking, fusion or reordering beyond the definition.  Pins: tests/test_oracle_pins.py
(brute-force index loops from oracle/brute_force.py on tiny shapes, closed forms S1-S4,
invariants I1/I1'/I2/I3/I6/S8, N=1; residual / batched / row-block forms against the brute
force) -- every function below is pinned there.
"""
from __future__ import annotations

from typing import Dict, Optional

import numpy as np

OUTGOING = 0
INCOMING = 1

_F = np.float64


def sigmoid(x: np.ndarray) -> np.ndarray:
    """1 / (1 + exp(-x)), evaluated without overflow for either sign of x."""
    x = np.asarray(x, dtype=_F)
    e = np.exp(-np.abs(x))
    return np.where(x >= 0, 1.0 / (1.0 + e), e / (1.0 + e))


def layer_norm(x: np.ndarray, gamma: np.ndarray, beta: np.ndarray, eps: float) -> np.ndarray:
    """LayerNorm over the last axis: (x - mean) / sqrt(var + eps) * gamma + beta, var = biased
    (divide by the channel count).  north_star "LayerNorm"; reading A6."""
    x = np.asarray(x, dtype=_F)
    mu = x.mean(axis=-1, keepdims=True)
    var = ((x - mu) ** 2).mean(axis=-1, keepdims=True)
    return (x - mu) / np.sqrt(var + eps) * np.asarray(gamma, _F) + np.asarray(beta, _F)


def _linear(x: np.ndarray, w: np.ndarray, b: Optional[np.ndarray]) -> np.ndarray:
    """torch.nn.Linear convention: y = x W^T + b, W is [out_features, in_features]."""
    x = np.asarray(x, _F)
    # leading dimensions flattened so that the product is ONE dense matmul (same definition,
    # same value per element; a 3-D @ 2-D numpy matmul would issue one small gemm per leading row)
    y = (x.reshape(-1, x.shape[-1]) @ np.asarray(w, _F).T).reshape(x.shape[:-1] + (np.shape(w)[0],))
    if b is not None:
        y = y + np.asarray(b, _F)
    return y


def gated_projection(zp: np.ndarray, mask: Optional[np.ndarray], w: np.ndarray,
                     b: Optional[np.ndarray], w_gate: np.ndarray,
                     b_gate: Optional[np.ndarray]) -> np.ndarray:
    """a = M * sigmoid(W_g z' + b_g) * (W z' + b)   (north_star; PAPER.md line 130
    "projections of the pair representation ... with element-wise gating")."""
    out = sigmoid(_linear(zp, w_gate, b_gate)) * _linear(zp, w, b)
    if mask is not None:
        out = np.asarray(mask, _F)[..., None] * out
    return out


def contraction(a: np.ndarray, b: np.ndarray, direction: int) -> np.ndarray:
    """PAPER.md Eq. 2-3 (lines 121-128).  a, b are [N, N, c]; returns o [N, N, c].

    outgoing: o[i, j, c] = sum_k a[i, k, c] * b[j, k, c]   -> per channel  A_c  B_c^T
    incoming: o[i, j, c] = sum_k a[k, i, c] * b[k, j, c]   -> per channel  A_c^T B_c
    """
    A = np.transpose(a, (2, 0, 1))      # [c, row, col]
    B = np.transpose(b, (2, 0, 1))
    if direction == OUTGOING:
        O = A @ np.transpose(B, (0, 2, 1))
    elif direction == INCOMING:
        O = np.transpose(A, (0, 2, 1)) @ B
    else:
        raise ValueError("direction must be 0 (outgoing) or 1 (incoming)")
    return np.transpose(O, (1, 2, 0))


def contraction_backward(d_o: np.ndarray, a: np.ndarray, b: np.ndarray, direction: int):
    """Gradients of Eq. 2-3 with respect to a and b, given d_o = dL/do
    (all [N, N, c]); the paper hand-writes every backward with the same algorithm as the forward
    (lines 92-96), SURVEY 8(f) NEXT-2.  Differentiating the definition term by term:

    outgoing  o[i,j] = sum_k a[i,k] b[j,k]:  d_a[i,k] = sum_j d_o[i,j] b[j,k]     (dO  B)
                                             d_b[j,k] = sum_i d_o[i,j] a[i,k]     (dO^T A)
    incoming  o[i,j] = sum_k a[k,i] b[k,j]:  d_a[k,i] = sum_j b[k,j] d_o[i,j]     (B  dO^T)
                                             d_b[k,j] = sum_i a[k,i] d_o[i,j]     (A  dO)
    per channel.  Returns (d_a, d_b), each [N, N, c].
    """
    G = np.transpose(np.asarray(d_o, _F), (2, 0, 1))
    A = np.transpose(np.asarray(a, _F), (2, 0, 1))
    B = np.transpose(np.asarray(b, _F), (2, 0, 1))
    T = lambda x: np.transpose(x, (0, 2, 1))
    if direction == OUTGOING:
        dA, dB = G @ B, T(G) @ A
    elif direction == INCOMING:
        dA, dB = B @ T(G), A @ G
    else:
        raise ValueError("direction must be 0 (outgoing) or 1 (incoming)")
    return np.transpose(dA, (1, 2, 0)), np.transpose(dB, (1, 2, 0))


def output_stage(o: np.ndarray, zp: np.ndarray, mask: Optional[np.ndarray],
                 p: Dict[str, np.ndarray], eps: float, mask_output: bool) -> np.ndarray:
    """out = [M *] sigmoid(W_g z' + b_g) * (W_o LayerNorm(o) + b_o)   (north_star)."""
    g = sigmoid(_linear(zp, p["w_g"], p.get("b_g")))
    y = _linear(layer_norm(o, p["ln_out_gamma"], p["ln_out_beta"], eps), p["w_o"], p.get("b_o"))
    out = g * y
    if mask_output and mask is not None:
        out = np.asarray(mask, _F)[..., None] * out
    return out


def trimul(z: np.ndarray, mask: Optional[np.ndarray], p: Dict[str, np.ndarray], direction: int,
           eps: float = 1e-5, mask_output: bool = True) -> np.ndarray:
    """Full op on z[N, N, c_z], pair mask M[N, N] (None = all ones) -> out[N, N, c_z] (fp64).

    `p` maps the names of paper_2603_14806_b200.synth.make_params to arrays; any bias may be
    absent / None (AF3's LinearNoBias).
    """
    z = np.asarray(z, _F)
    zp = layer_norm(z, p["ln_in_gamma"], p["ln_in_beta"], eps)
    a = gated_projection(zp, mask, p["w_a"], p.get("b_a"), p["w_a_gate"], p.get("b_a_gate"))
    b = gated_projection(zp, mask, p["w_b"], p.get("b_b"), p["w_b_gate"], p.get("b_b_gate"))
    o = contraction(a, b, direction)
    return output_stage(o, zp, mask, p, eps, mask_output)


def trimul_residual(z: np.ndarray, mask: Optional[np.ndarray], p: Dict[str, np.ndarray],
                    direction: int, eps: float = 1e-5, mask_output: bool = True) -> np.ndarray:
    """The paper's own form of the update, PAPER.md lines 121-128 (Eq. 2-3 are written
    "z_nm += ..."): z + trimul(z).  SURVEY 8(f) NEXT-1; c_hidden need not equal c_z, the update
    always has c_z channels."""
    z = np.asarray(z, _F)
    return z + trimul(z, mask, p, direction, eps=eps, mask_output=mask_output)


def trimul_batched(z: np.ndarray, mask: Optional[np.ndarray], p: Dict[str, np.ndarray],
                   direction: int, eps: float = 1e-5, mask_output: bool = True,
                   residual: bool = False) -> np.ndarray:
    """z[B, N, N, c_z] (z in R^{B x N x N x D}), pair mask [B, N, N] or None:
    the batch elements are independent problems with shared parameters."""
    f = trimul_residual if residual else trimul
    return np.stack([f(z[b], None if mask is None else mask[b], p, direction, eps=eps,
                       mask_output=mask_output) for b in range(z.shape[0])])


def trimul_subgrid(z_a: np.ndarray, mask_a: Optional[np.ndarray],
                   z_b: np.ndarray, mask_b: Optional[np.ndarray],
                   z_ij: np.ndarray, mask_ij: Optional[np.ndarray],
                   p: Dict[str, np.ndarray], eps: float = 1e-5,
                   mask_output: bool = True) -> np.ndarray:
    """Exact out[I x J] (full sums over k) from only the slices of z the definition touches.

    For index sets I, J the caller passes, in (row, k) order:
        outgoing:  z_a = z[I, :, :]            z_b = z[J, :, :]            (a_ik, b_jk)
        incoming:  z_a = z[:, I, :] swapped    z_b = z[:, J, :] swapped    (a_ki, b_kj)
    to [|I|, N, c_z] / [|J|, N, c_z] (and the matching pair-mask slices), plus
    z_ij = z[I][:, J] ([|I|, |J|, c_z]) for the output gate.  With the slices in that order
    both directions are the same formula  o_ij = sum_k a'_ik * b'_jk  -- PAPER.md line 132:
    the variants "differ only in which operand is transposed".
    """
    zpa = layer_norm(z_a, p["ln_in_gamma"], p["ln_in_beta"], eps)
    zpb = layer_norm(z_b, p["ln_in_gamma"], p["ln_in_beta"], eps)
    a = gated_projection(zpa, mask_a, p["w_a"], p.get("b_a"), p["w_a_gate"], p.get("b_a_gate"))
    b = gated_projection(zpb, mask_b, p["w_b"], p.get("b_b"), p["w_b_gate"], p.get("b_b_gate"))
    A = np.transpose(a, (2, 0, 1))                    # [c, |I|, N]
    B = np.transpose(b, (2, 0, 1))                    # [c, |J|, N]
    o = np.transpose(A @ np.transpose(B, (0, 2, 1)), (1, 2, 0))   # [|I|, |J|, c]
    zp_ij = layer_norm(z_ij, p["ln_in_gamma"], p["ln_in_beta"], eps)
    return output_stage(o, zp_ij, mask_ij, p, eps, mask_output)


def projections(z: np.ndarray, mask: Optional[np.ndarray], p: Dict[str, np.ndarray],
                eps: float = 1e-5):
    """(a, b) = the two gated, masked projections of LayerNorm(z) (north_star),
    for z of any leading shape [..., c_z] and a mask of that leading shape: every pair is
    independent, so a caller may evaluate a tensor too large for host memory slice by slice."""
    zp = layer_norm(z, p["ln_in_gamma"], p["ln_in_beta"], eps)
    a = gated_projection(zp, mask, p["w_a"], p.get("b_a"), p["w_a_gate"], p.get("b_a_gate"))
    b = gated_projection(zp, mask, p["w_b"], p.get("b_b"), p["w_b_gate"], p.get("b_b_gate"))
    return a, b


def trimul_rowblock(a: np.ndarray, b: np.ndarray, z_rows: np.ndarray,
                    mask_rows: Optional[np.ndarray], p: Dict[str, np.ndarray], direction: int,
                    i0: int, i1: int, eps: float = 1e-5, mask_output: bool = True) -> np.ndarray:
    """Exact out[i0:i1, :, :] of the full op with bounded memory (whole-tensor parity at N = 4096,
    where out alone is 17 GB in fp64).  `a`, `b` [N, N, c] are the projections of the WHOLE z
    (from `projections`); z_rows = z[i0:i1], mask_rows = M[i0:i1] feed the output gate / mask.

    PAPER.md Eq. 2-3 (lines 121-128) restricted to output rows i0..i1-1, nothing else changed:
      outgoing: o[i, j] = sum_k a[i, k] b[j, k]   needs a's ROWS    i0:i1 and all of b
      incoming: o[i, j] = sum_k a[k, i] b[k, j]   needs a's COLUMNS i0:i1 and all of b
    followed by the same output stage as `trimul`."""
    B = np.transpose(np.asarray(b, _F), (2, 0, 1))                       # [c, row, col]
    if direction == OUTGOING:
        A = np.transpose(np.asarray(a[i0:i1], _F), (2, 0, 1))            # [c, i, k]
        O = A @ np.transpose(B, (0, 2, 1))                               # sum_k a[i,k] b[j,k]
    elif direction == INCOMING:
        A = np.transpose(np.asarray(a[:, i0:i1], _F), (2, 1, 0))         # [c, i, k] = a[k, i]
        O = A @ B                                                        # sum_k a[k,i] b[k,j]
    else:
        raise ValueError("direction must be 0 (outgoing) or 1 (incoming)")
    o = np.transpose(O, (1, 2, 0))                                       # [i1 - i0, N, c]
    zp = layer_norm(z_rows, p["ln_in_gamma"], p["ln_in_beta"], eps)
    return output_stage(o, zp, mask_rows, p, eps, mask_output)


# ------------------------------------------------------------------------------------------------
# Backward pass.  PAPER.md lines 92-96 (section 3.1): every Fold-CP module
# hand-writes its forward AND backward with the same algorithm.  The functions below are the chain
# rule applied to the definition above, one forward line at a time in reverse order; nothing is
# fused or reordered.  Pins (tests/test_oracle_pins.py): central finite differences of `trimul` for
# every input and parameter, the adjoint identity <d_out, J u> = <J^T d_out, u>, and a scalar-loop
# Jacobian for the LayerNorm backward.
# ------------------------------------------------------------------------------------------------
def layer_norm_backward(d_y: np.ndarray, x: np.ndarray, gamma: np.ndarray, eps: float):
    """Backward of y = (x - mean) / sqrt(var + eps) * gamma + beta over the last axis (biased var).
    With xh = (x - mean) / sqrt(var + eps) and d_xh = d_y * gamma:
        d_x     = (d_xh - mean(d_xh) - xh * mean(d_xh * xh)) / sqrt(var + eps)
        d_gamma = sum over rows of d_y * xh        d_beta = sum over rows of d_y
    Returns (d_x, d_gamma, d_beta)."""
    x = np.asarray(x, _F)
    d_y = np.asarray(d_y, _F)
    mu = x.mean(axis=-1, keepdims=True)
    var = ((x - mu) ** 2).mean(axis=-1, keepdims=True)
    rstd = 1.0 / np.sqrt(var + eps)
    xh = (x - mu) * rstd
    d_xh = d_y * np.asarray(gamma, _F)
    d_x = (d_xh - d_xh.mean(axis=-1, keepdims=True)
           - xh * (d_xh * xh).mean(axis=-1, keepdims=True)) * rstd
    lead = tuple(range(x.ndim - 1))
    return d_x, (d_y * xh).sum(axis=lead), d_y.sum(axis=lead)


def _linear_backward(d_y: np.ndarray, x: np.ndarray, w: np.ndarray):
    """Backward of y = x W^T + b:  d_x = d_y W,  d_W = d_y^T x,  d_b = sum of d_y (rows flattened)."""
    d2 = np.asarray(d_y, _F).reshape(-1, d_y.shape[-1])
    x2 = np.asarray(x, _F).reshape(-1, x.shape[-1])
    d_x = (d2 @ np.asarray(w, _F)).reshape(x.shape)
    return d_x, d2.T @ x2, d2.sum(axis=0)


def trimul_backward(d_out: np.ndarray, z: np.ndarray, mask: Optional[np.ndarray],
                    p: Dict[str, np.ndarray], direction: int, eps: float = 1e-5,
                    mask_output: bool = True, residual: bool = False):
    """Gradients of L = <d_out, trimul(z)> (or of the residual form z + trimul(z)).

    Returns (d_z [N, N, c_z], grads) where grads maps every parameter name of `p` (the six weight
    matrices, the biases that are present, both LayerNorm gammas and betas) to its gradient.
    The forward intermediates are recomputed here exactly as `trimul` computes them."""
    z = np.asarray(z, _F)
    d_out = np.asarray(d_out, _F)
    Mf = None if mask is None else np.asarray(mask, _F)[..., None]
    # ---- forward, keeping the intermediates
    zp = layer_norm(z, p["ln_in_gamma"], p["ln_in_beta"], eps)
    pa, ga = _linear(zp, p["w_a"], p.get("b_a")), _linear(zp, p["w_a_gate"], p.get("b_a_gate"))
    pb, gb = _linear(zp, p["w_b"], p.get("b_b")), _linear(zp, p["w_b_gate"], p.get("b_b_gate"))
    sa, sb = sigmoid(ga), sigmoid(gb)
    a, b = sa * pa, sb * pb
    if Mf is not None:
        a, b = Mf * a, Mf * b
    g = sigmoid(_linear(zp, p["w_g"], p.get("b_g")))
    o = contraction(a, b, direction)
    on = layer_norm(o, p["ln_out_gamma"], p["ln_out_beta"], eps)
    y = _linear(on, p["w_o"], p.get("b_o"))
    # ---- out = [M] g y
    d_gy = d_out if (Mf is None or not mask_output) else d_out * Mf
    d_y = d_gy * g
    d_gg = d_gy * y * g * (1.0 - g)                       # through g = sigmoid(gg)
    grads: Dict[str, np.ndarray] = {}
    d_on, grads["w_o"], db = _linear_backward(d_y, on, p["w_o"])
    if p.get("b_o") is not None:
        grads["b_o"] = db
    d_o, grads["ln_out_gamma"], grads["ln_out_beta"] = layer_norm_backward(d_on, o, p["ln_out_gamma"], eps)
    # ---- Eq. 2-3
    d_a, d_b = contraction_backward(d_o, a, b, direction)
    if Mf is not None:
        d_a, d_b = d_a * Mf, d_b * Mf
    # ---- a = M sigmoid(ga) pa, b likewise
    d_zp, grads["w_g"], db = _linear_backward(d_gg, zp, p["w_g"])
    if p.get("b_g") is not None:
        grads["b_g"] = db
    for d_t, s_t, p_t, wn, bn, gwn, gbn in ((d_a, sa, pa, "w_a", "b_a", "w_a_gate", "b_a_gate"),
                                            (d_b, sb, pb, "w_b", "b_b", "w_b_gate", "b_b_gate")):
        d_p = d_t * s_t
        d_gate = d_t * p_t * s_t * (1.0 - s_t)
        dx, grads[wn], db = _linear_backward(d_p, zp, p[wn])
        if p.get(bn) is not None:
            grads[bn] = db
        d_zp = d_zp + dx
        dx, grads[gwn], db = _linear_backward(d_gate, zp, p[gwn])
        if p.get(gbn) is not None:
            grads[gbn] = db
        d_zp = d_zp + dx
    d_z, grads["ln_in_gamma"], grads["ln_in_beta"] = layer_norm_backward(d_zp, z, p["ln_in_gamma"], eps)
    if residual:
        d_z = d_z + d_out
    return d_z, grads


# ------------------------------------------------------------------------------------------------
# The paper's distributed form.  PAPER.md lines 132-134, section 3.3 "Sharding
# and algorithm": "The pair representation is tiled as (N/sqrt(P))^2 blocks.  One operand is
# transposed across the 2D grid to align the contracted index with the ring shift direction.  The
# algorithm then proceeds in a Cannon-style ring: in each of sqrt(P) steps, ranks perform a local
# batched matrix multiplication between resident blocks of a and b while simultaneously initiating
# asynchronous P2P transfers to circulate a along rows and b along columns.  Partial results
# accumulate into the output block.  The outgoing and incoming variants differ only in which operand
# is transposed" (Fig. 2b; Table 1, line 83).
#
# Written out step by step on a simulated g x g grid (rank (r, c) owns block (r, c) of every pair
# tensor).  The paper names Cannon's algorithm without restating its initial alignment; the reading
# taken (A23) is the textbook one: after the grid transpose, the row-circulating operand
# of grid row r is pre-shifted by r and the column-circulating operand of grid column c by c, so
# that in step s rank (r, c) multiplies the two blocks with contracted block index
# q = (r + c + s) mod g; then both circulate by one position per step.
# ------------------------------------------------------------------------------------------------
def cannon_schedule(grid: int, direction: int):
    """Which blocks rank (r, c) multiplies in step s.  Returns a dict
    {(r, c): [((ar, ac), (br, bc)) for s in range(grid)]} of block coordinates of a and of b.
      outgoing: o_rc = sum_q a_(r,q) b_(c,q)^T   -> b is the operand transposed across the grid
      incoming: o_rc = sum_q a_(q,r)^T b_(q,c)   -> a is the operand transposed across the grid"""
    sched = {}
    for r in range(grid):
        for c in range(grid):
            steps = []
            for s_ in range(grid):
                q = (r + c + s_) % grid
                steps.append((((r, q), (c, q)) if direction == OUTGOING else ((q, r), (q, c))))
            sched[(r, c)] = steps
    return sched


def contraction_cannon(a: np.ndarray, b: np.ndarray, direction: int, grid: int) -> np.ndarray:
    """Eq. 2-3 computed the paper's way on a simulated grid x grid mesh; equals `contraction`.
    a, b [N, N, c] with N divisible by grid (the paper's tiling).  Every data movement of the
    algorithm is carried out explicitly on per-rank block dictionaries."""
    a = np.asarray(a, _F)
    b = np.asarray(b, _F)
    N = a.shape[0]
    g = int(grid)
    if direction not in (OUTGOING, INCOMING):
        raise ValueError("direction must be 0 (outgoing) or 1 (incoming)")
    if N % g != 0:
        raise ValueError("N must be divisible by the grid size")
    nb = N // g
    blk = lambda t, r, c: t[r * nb:(r + 1) * nb, c * nb:(c + 1) * nb]
    ranks = [(r, c) for r in range(g) for c in range(g)]
    # 0. tiling: rank (r, c) owns block (r, c) of a and of b
    A = {rc: blk(a, *rc).copy() for rc in ranks}
    Bm = {rc: blk(b, *rc).copy() for rc in ranks}
    # 1. one operand is transposed across the grid: rank (r, c) receives the block of rank (c, r)
    if direction == OUTGOING:
        Bm = {(r, c): Bm[(c, r)] for (r, c) in ranks}       # rank (r, c) now holds b_(c, r)
    else:
        A = {(r, c): A[(c, r)] for (r, c) in ranks}         # rank (r, c) now holds a_(c, r)
    # 2. Cannon's initial alignment (reading A23).  After step 1, in BOTH directions the contracted
    #    block index of the a block a rank holds varies along its grid row and that of its b block
    #    along its grid column:
    #      outgoing: rank (r, c) holds a_(r, c) and b_(c, r)    (contracted index: c for a, r for b)
    #      incoming: rank (r, c) holds a_(c, r) and b_(r, c)    (contracted index: c for a, r for b)
    #    which is why "a circulates along rows and b along columns" whatever the direction.
    A = {(r, c): A[(r, (c + r) % g)] for (r, c) in ranks}   # row r of the grid pre-shifted by r
    Bm = {(r, c): Bm[((r + c) % g, c)] for (r, c) in ranks} # column c of the grid pre-shifted by c
    out = {rc: np.zeros((nb, nb, a.shape[2]), _F) for rc in ranks}
    for _step in range(g):
        # local batched matrix multiplication between the resident blocks, accumulated
        for rc in ranks:
            out[rc] += contraction(A[rc], Bm[rc], direction)
        # circulate a along rows and b along columns by one position
        A = {(r, c): A[(r, (c + 1) % g)] for (r, c) in ranks}
        Bm = {(r, c): Bm[((r + 1) % g, c)] for (r, c) in ranks}
    o = np.empty_like(a)
    for (r, c) in ranks:
        o[r * nb:(r + 1) * nb, c * nb:(c + 1) * nb] = out[(r, c)]
    return o


def trimul_cannon(z: np.ndarray, mask: Optional[np.ndarray], p: Dict[str, np.ndarray],
                  direction: int, grid: int, eps: float = 1e-5, mask_output: bool = True) -> np.ndarray:
    """The full op with the contraction done the paper's distributed way.  LayerNorm, projections,
    gates and the output stage act on each pair independently, so every rank applies them to its own
    block of z; only Eq. 2-3 need the ring."""
    z = np.asarray(z, _F)
    zp = layer_norm(z, p["ln_in_gamma"], p["ln_in_beta"], eps)
    a, b = projections(z, mask, p, eps)
    o = contraction_cannon(a, b, direction, grid)
    return output_stage(o, zp, mask, p, eps, mask_output)


def flops(N: int, c_z: int, c_hidden: int) -> float:
    """Counted FLOPs of one call: contraction 2 c N^3 + five
    projections 2 N^2 c_z (4c + c_z) + output projection 2 N^2 c c_z."""
    return 2.0 * c_hidden * N ** 3 + 2.0 * N * N * c_z * (4 * c_hidden + c_z) \
        + 2.0 * N * N * c_hidden * c_z
