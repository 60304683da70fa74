"""fp64 CPU oracle of triangle attention (starting node = over rows, ending node = over columns).

TEST INFRASTRUCTURE -- NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline leg may import this package.  It shares no code with the CUDA path and never imports it.

What it computes (plain definition, numpy fp64):

  PAPER.md lines 98-115, section 3.2, Eq. 1: "multi-head attention over the rows (or columns) of the
  pair tensor, with an additive triangular bias derived from the same representation":
      Q, K, V = proj(z),   output = softmax(Q K^T / sqrt(d) + tri_bias(z) + mask_bias) V
  "The triangular bias operates along an axis orthogonal to the padding mask ... all three axes
  {i, j, k}".  The paper leaves out the LayerNorm, the gate and the output projection; they are
  those of AF3 supplementary Alg. 14 / 15 (restated from the published definition; DESIGN.md
  readings T1-T4):

      z'      = LayerNorm(z)                                   over c_z, biased variance, eps in sqrt
      q, k, v = W_q z', W_k z', W_v z'                          [N, N, H, c]   no biases
      t       = W_t z'                                          [N, N, H]      the triangular bias
      g       = sigmoid(W_g z')                                 [N, N, H, c]
    starting node (rows):     s_ijk = q_ij . k_ik / sqrt(c) + t_jk + mb_ik ,   o_ij = g_ij * sum_k softmax_k(s_ijk) v_ik
    ending node (columns):    s_ijk = q_ij . k_kj / sqrt(c) + t_ki + mb_kj ,   o_ij = g_ij * sum_k softmax_k(s_ijk) v_kj
      out_ij  = W_o concat_h(o_ij)                              [N, N, c_z]
  with mb = -1e9 * (1 - M) for a pair mask M in {0, 1} (the key position's mask).

A library primitive (numpy einsum / matmul) serves as the dense step; nothing is blocked, fused or
reordered beyond the definition (the softmax subtracts the row maximum, which changes no value).
Pins: tests/test_triattn_oracle_pins.py (scalar loops from `triattn_brute` below on tiny shapes, rows
of the attention weights sum to one, the ending node is the starting node on the transposed input,
masked keys get exactly zero weight, uniform attention when q = 0 and t = 0, token permutation).
"""
from __future__ import annotations

import math
from typing import Dict, Optional

import numpy as np

STARTING = 0
ENDING = 1
MASK_BIAS = -1.0e9


def _layer_norm(x, gamma, beta, eps):
    mu = x.mean(axis=-1, keepdims=True)
    var = ((x - mu) ** 2).mean(axis=-1, keepdims=True)
    return (x - mu) / np.sqrt(var + eps) * gamma + beta


def projections(z, p, n_heads, eps=1e-5):
    """(q, k, v, g) as [N, N, H, c] and t as [N, N, H] from z [N, N, c_z] (Alg. 14 lines 1-4)."""
    z = np.asarray(z, dtype=np.float64)
    N = z.shape[0]
    zp = _layer_norm(z, p["ln_gamma"], p["ln_beta"], eps)
    H = n_heads
    c = p["w_q"].shape[0] // H
    q = (zp @ p["w_q"].T).reshape(N, N, H, c)
    k = (zp @ p["w_k"].T).reshape(N, N, H, c)
    v = (zp @ p["w_v"].T).reshape(N, N, H, c)
    g = 1.0 / (1.0 + np.exp(-(zp @ p["w_g"].T))).reshape(N, N, H, c)
    t = zp @ p["w_t"].T
    return q, k, v, g, t


def attention_weights(q, k, t, mask, node):
    """a[i, j, k, h] = softmax over k of the scores of Eq. 1."""
    N, _, H, c = q.shape
    mb = np.zeros((N, N)) if mask is None else MASK_BIAS * (1.0 - np.asarray(mask, dtype=np.float64))
    if node == STARTING:
        s = np.einsum("ijhc,ikhc->ijkh", q, k) / math.sqrt(c)
        s = s + t[None, :, :, :] + mb[:, None, :, None]          # t_jk , mb_ik
    else:
        s = np.einsum("ijhc,kjhc->ijkh", q, k) / math.sqrt(c)
        s = s + np.transpose(t, (1, 0, 2))[:, None, :, :] + mb.T[None, :, :, None]   # t_ki , mb_kj
    s = s - s.max(axis=2, keepdims=True)
    e = np.exp(s)
    return e / e.sum(axis=2, keepdims=True)


def triangle_attention(z, mask, p: Dict[str, np.ndarray], node: int, n_heads: int = 4,
                       eps: float = 1e-5):
    """Full op: z [N, N, c_z], pair mask [N, N] in {0, 1} or None -> out [N, N, c_z] (fp64)."""
    q, k, v, g, t = projections(z, p, n_heads, eps)
    a = attention_weights(q, k, t, mask, node)
    if node == STARTING:
        o = np.einsum("ijkh,ikhc->ijhc", a, v)
    else:
        o = np.einsum("ijkh,kjhc->ijhc", a, v)
    o = g * o
    N = o.shape[0]
    return o.reshape(N, N, -1) @ p["w_o"].T


def flops(N: int, c_z: int, n_heads: int, c_head: int) -> float:
    """Counted FLOPs: QK^T and PV (2 * 2 N^3 H c) + the five projections, the bias and the output
    projection (matmul FLOPs only, like the triangle multiplication's count)."""
    hc = n_heads * c_head
    return 4.0 * N ** 3 * hc + 2.0 * N * N * c_z * (4 * hc + n_heads) + 2.0 * N * N * hc * c_z


# ------------------------------------------------------------------------------------------------
# brute force: scalar Python loops, `math` only -- used ONLY to pin the functions above on tiny shapes
# ------------------------------------------------------------------------------------------------
def triattn_brute(z, mask, p, node, n_heads, eps=1e-5):
    """z: nested lists [N][N][c_z]; mask [N][N] or None; p: dict of nested lists. Returns nested lists."""
    N, cz = len(z), len(z[0][0])
    H = n_heads
    c = len(p["w_q"]) // H

    def ln(vv):
        mu = sum(vv) / cz
        var = sum((x - mu) ** 2 for x in vv) / cz
        r = 1.0 / math.sqrt(var + eps)
        return [(vv[d] - mu) * r * p["ln_gamma"][d] + p["ln_beta"][d] for d in range(cz)]

    def mv(w, x):
        return [sum(w[r][d] * x[d] for d in range(len(x))) for r in range(len(w))]

    zp = [[ln(z[i][j]) for j in range(N)] for i in range(N)]
    Q = [[mv(p["w_q"], zp[i][j]) for j in range(N)] for i in range(N)]
    K = [[mv(p["w_k"], zp[i][j]) for j in range(N)] for i in range(N)]
    V = [[mv(p["w_v"], zp[i][j]) for j in range(N)] for i in range(N)]
    G = [[[1.0 / (1.0 + math.exp(-x)) for x in mv(p["w_g"], zp[i][j])] for j in range(N)] for i in range(N)]
    T = [[mv(p["w_t"], zp[i][j]) for j in range(N)] for i in range(N)]
    out = [[[0.0] * cz for _ in range(N)] for _ in range(N)]
    for i in range(N):
        for j in range(N):
            o = [0.0] * (H * c)
            for h in range(H):
                s = []
                for k in range(N):
                    if node == STARTING:
                        kk, tb, m = K[i][k], T[j][k][h], (1.0 if mask is None else mask[i][k])
                    else:
                        kk, tb, m = K[k][j], T[k][i][h], (1.0 if mask is None else mask[k][j])
                    dot = sum(Q[i][j][h * c + d] * kk[h * c + d] for d in range(c))
                    s.append(dot / math.sqrt(c) + tb + MASK_BIAS * (1.0 - m))
                mx = max(s)
                e = [math.exp(x - mx) for x in s]
                den = sum(e)
                for d in range(c):
                    acc = 0.0
                    for k in range(N):
                        vv = V[i][k] if node == STARTING else V[k][j]
                        acc += e[k] / den * vv[h * c + d]
                    o[h * c + d] = G[i][j][h * c + d] * acc
            out[i][j] = mv(p["w_o"], o)
    return out
