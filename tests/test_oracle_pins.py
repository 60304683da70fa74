"""Pins of the fp64 oracle against things other than itself (run with -m "not gpu").

Each test is chosen so that a plausible mistake in oracle/trimul_oracle.py (dropped term,
wrong sign or index, transposed operand, mask in the wrong place, unbiased variance, ...)
fails at least one of them.  Names follow SURVEY.md section 8(c).
"""
import math

import numpy as np
import pytest

from oracle import brute_force
from oracle import trimul_oracle as orc

OUT, INC = orc.OUTGOING, orc.INCOMING


def rand_params(rng, c_z, c, bias=True):
    p = {
        "ln_in_gamma": 1 + 0.1 * rng.standard_normal(c_z), "ln_in_beta": 0.1 * rng.standard_normal(c_z),
        "w_a": rng.standard_normal((c, c_z)) / math.sqrt(c_z),
        "w_a_gate": rng.standard_normal((c, c_z)) / math.sqrt(c_z),
        "w_b": rng.standard_normal((c, c_z)) / math.sqrt(c_z),
        "w_b_gate": rng.standard_normal((c, c_z)) / math.sqrt(c_z),
        "w_g": rng.standard_normal((c_z, c_z)) / math.sqrt(c_z),
        "ln_out_gamma": 1 + 0.1 * rng.standard_normal(c), "ln_out_beta": 0.1 * rng.standard_normal(c),
        "w_o": rng.standard_normal((c_z, c)) / math.sqrt(c),
    }
    if bias:
        for k, n in (("b_a", c), ("b_a_gate", c), ("b_b", c), ("b_b_gate", c), ("b_g", c_z), ("b_o", c_z)):
            p[k] = 0.3 * rng.standard_normal(n)
    return p


def swap_ab(p):
    q = dict(p)
    for x, y in (("w_a", "w_b"), ("w_a_gate", "w_b_gate"), ("b_a", "b_b"), ("b_a_gate", "b_b_gate")):
        if x in p:
            q[x], q[y] = p[y], p[x]
    return q


def tolist(p):
    return {k: np.asarray(v).tolist() for k, v in p.items()}


def relerr(x, y):
    return np.linalg.norm(x - y) / max(np.linalg.norm(y), 1e-300)


# ----------------------------------------------------------------------------------------
# brute force (pure-Python scalar loops) on tiny shapes, both directions, general pair mask
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,c_z,c", [(1, 4, 3), (2, 4, 3), (3, 8, 8), (5, 4, 8), (8, 8, 3)])
@pytest.mark.parametrize("direction", [OUT, INC])
@pytest.mark.parametrize("mask_output", [True, False])
def test_brute_force(N, c_z, c, direction, mask_output):
    rng = np.random.default_rng(100 * N + 10 * c_z + c + direction)
    z = rng.standard_normal((N, N, c_z))
    M = (rng.random((N, N)) > 0.3).astype(np.float64)       # general, non-symmetric pair mask
    p = rand_params(rng, c_z, c)
    got = orc.trimul(z, M, p, direction, mask_output=mask_output)
    ref = np.array(brute_force.trimul_brute(z.tolist(), M.tolist(), tolist(p), direction,
                                            mask_output=mask_output))
    assert got.shape == (N, N, c_z)
    assert relerr(got, ref) < 1e-12


@pytest.mark.parametrize("direction", [OUT, INC])
def test_residual_and_batched_forms_against_brute_force(direction):
    """PAPER.md lines 121-128 write the update as `z_nm += ...`; line 130 carries a batch
    dimension.  Pinned against the scalar loops: residual = z + brute-force update, element by
    element; batched = the brute force applied to every batch element separately."""
    rng = np.random.default_rng(31 + direction)
    Bn, N, c_z, c = 2, 4, 8, 3
    z = rng.standard_normal((Bn, N, N, c_z))
    M = (rng.random((Bn, N, N)) > 0.3).astype(np.float64)
    p = rand_params(rng, c_z, c)
    upd = [np.array(brute_force.trimul_brute(z[b].tolist(), M[b].tolist(), tolist(p), direction))
           for b in range(Bn)]
    for b in range(Bn):
        got = orc.trimul_residual(z[b], M[b], p, direction)
        want = np.array([[[z[b, i, j, ch] + upd[b][i, j, ch] for ch in range(c_z)]
                          for j in range(N)] for i in range(N)])
        assert relerr(got, want) < 1e-12
    got = orc.trimul_batched(z, M, p, direction)
    assert got.shape == (Bn, N, N, c_z) and relerr(got, np.stack(upd)) < 1e-12
    got = orc.trimul_batched(z, M, p, direction, residual=True)
    assert relerr(got, z + np.stack(upd)) < 1e-12
    # a zero update (W_o = 0, b_o = 0: closed form S4) leaves exactly z
    q = dict(p); q["w_o"] = np.zeros_like(p["w_o"]); q["b_o"] = np.zeros_like(p["b_o"])
    assert np.array_equal(orc.trimul_residual(z[0], M[0], q, direction), z[0])


@pytest.mark.parametrize("direction", [OUT, INC])
def test_contraction_backward_against_loops_and_directional_derivative(direction):
    """d_a, d_b of Eq. 2-3: (i) literal index loops of the differentiated definition; (ii) the
    forward contraction is bilinear, so <d_o, o(a + u, b) - o(a, b)> = <d_a, u> exactly (and the
    same for b) -- a wrong index or a transposed operand breaks it."""
    rng = np.random.default_rng(77 + direction)
    N, c = 5, 3
    a, b, g = (rng.standard_normal((N, N, c)) for _ in range(3))
    da, db = orc.contraction_backward(g, a, b, direction)
    ra, rb = np.zeros_like(a), np.zeros_like(b)
    for ch in range(c):
        for i in range(N):
            for j in range(N):
                for k in range(N):
                    if direction == OUT:      # o[i,j] += a[i,k] b[j,k]
                        ra[i, k, ch] += g[i, j, ch] * b[j, k, ch]
                        rb[j, k, ch] += g[i, j, ch] * a[i, k, ch]
                    else:                     # o[i,j] += a[k,i] b[k,j]
                        ra[k, i, ch] += g[i, j, ch] * b[k, j, ch]
                        rb[k, j, ch] += g[i, j, ch] * a[k, i, ch]
    assert relerr(da, ra) < 1e-12 and relerr(db, rb) < 1e-12
    u, v = rng.standard_normal(a.shape), rng.standard_normal(b.shape)
    o0 = orc.contraction(a, b, direction)
    lhs_a = np.sum(g * (orc.contraction(a + u, b, direction) - o0))
    lhs_b = np.sum(g * (orc.contraction(a, b + v, direction) - o0))
    assert abs(lhs_a - np.sum(da * u)) < 1e-10 * max(1.0, abs(lhs_a))
    assert abs(lhs_b - np.sum(db * v)) < 1e-10 * max(1.0, abs(lhs_b))


def test_brute_force_no_bias_no_mask_soft_mask():
    rng = np.random.default_rng(7)
    N, c_z, c = 4, 8, 4
    z = rng.standard_normal((N, N, c_z))
    p = rand_params(rng, c_z, c, bias=False)
    for direction in (OUT, INC):
        got = orc.trimul(z, None, p, direction)
        ref = np.array(brute_force.trimul_brute(z.tolist(), None, tolist(p), direction))
        assert relerr(got, ref) < 1e-12
        Ms = rng.random((N, N))                              # soft (non 0/1) mask: multiplied as-is (A22)
        got = orc.trimul(z, Ms, p, direction)
        ref = np.array(brute_force.trimul_brute(z.tolist(), Ms.tolist(), tolist(p), direction))
        assert relerr(got, ref) < 1e-12


def test_none_bias_equals_zero_bias_bitwise():
    rng = np.random.default_rng(8)
    N, c_z, c = 5, 8, 8
    z = rng.standard_normal((N, N, c_z))
    p = rand_params(rng, c_z, c, bias=False)
    pz = dict(p)
    for k, n in (("b_a", c), ("b_a_gate", c), ("b_b", c), ("b_b_gate", c), ("b_g", c_z), ("b_o", c_z)):
        pz[k] = np.zeros(n)
    for d in (OUT, INC):
        assert np.array_equal(orc.trimul(z, None, p, d), orc.trimul(z, None, pz, d))


# ----------------------------------------------------------------------------------------
# contraction alone: Eq. 2-3 against scalar loops, I1' (swapped layouts), library matmul (S5)
# ----------------------------------------------------------------------------------------
def test_contraction_definition_loops():
    rng = np.random.default_rng(1)
    N, c = 6, 5
    a = rng.standard_normal((N, N, c))
    b = rng.standard_normal((N, N, c))
    o_out = np.zeros((N, N, c))
    o_in = np.zeros((N, N, c))
    for i in range(N):
        for j in range(N):
            for k in range(N):
                o_out[i, j] += a[i, k] * b[j, k]
                o_in[i, j] += a[k, i] * b[k, j]
    assert np.allclose(orc.contraction(a, b, OUT), o_out, rtol=0, atol=1e-13)
    assert np.allclose(orc.contraction(a, b, INC), o_in, rtol=0, atol=1e-13)
    # a wrong reading (transposing only one operand) must NOT pass
    assert not np.allclose(orc.contraction(a, b, OUT), o_in, atol=1e-3)


def test_I1prime_contraction_swapped_layouts():
    rng = np.random.default_rng(2)
    N, c = 7, 4
    a = rng.standard_normal((N, N, c))
    b = rng.standard_normal((N, N, c))
    aT, bT = np.transpose(a, (1, 0, 2)), np.transpose(b, (1, 0, 2))
    assert np.allclose(orc.contraction(a, b, INC), orc.contraction(aT, bT, OUT), rtol=0, atol=1e-13)


def test_S5_reduces_to_dense_matmul():
    """Gates saturated (sigmoid(+40) == 1 in fp64): a, b are affine maps of z' and each channel of
    o is a textbook dense matrix product; checked through gamma_out-scaled pre-LN quantities."""
    rng = np.random.default_rng(3)
    N, c_z, c = 9, 8, 6
    z = rng.standard_normal((N, N, c_z))
    p = rand_params(rng, c_z, c)
    for k in ("w_a_gate", "w_b_gate"):
        p[k] = np.zeros_like(p[k])
    p["b_a_gate"] = np.full(c, 40.0)
    p["b_b_gate"] = np.full(c, 40.0)
    zp = orc.layer_norm(z, p["ln_in_gamma"], p["ln_in_beta"], 1e-5)
    a = orc.gated_projection(zp, None, p["w_a"], p["b_a"], p["w_a_gate"], p["b_a_gate"])
    b = orc.gated_projection(zp, None, p["w_b"], p["b_b"], p["w_b_gate"], p["b_b_gate"])
    assert np.allclose(a, zp @ p["w_a"].T + p["b_a"], rtol=1e-15, atol=1e-15)
    for ch in range(c):
        A, B = a[:, :, ch], b[:, :, ch]
        assert np.allclose(orc.contraction(a, b, OUT)[:, :, ch], np.einsum("ik,jk->ij", A, B), atol=1e-12)
        assert np.allclose(orc.contraction(a, b, INC)[:, :, ch], np.einsum("ki,kj->ij", A, B), atol=1e-12)


# ----------------------------------------------------------------------------------------
# invariants
# ----------------------------------------------------------------------------------------
def test_I1_direction_identity_needs_ab_swap():
    """incoming(z, M; theta) = T(outgoing(Tz, TM; theta with a<->b swapped)); the naive form of
    north_star (no swap) is false for distinct a/b parameters (reading A10)."""
    rng = np.random.default_rng(4)
    N, c_z, c = 6, 8, 5
    z = rng.standard_normal((N, N, c_z))
    M = (rng.random((N, N)) > 0.3).astype(np.float64)
    p = rand_params(rng, c_z, c)
    zT, MT = np.transpose(z, (1, 0, 2)), M.T
    inc = orc.trimul(z, M, p, INC)
    good = np.transpose(orc.trimul(zT, MT, swap_ab(p), OUT), (1, 0, 2))
    naive = np.transpose(orc.trimul(zT, MT, p, OUT), (1, 0, 2))
    assert relerr(good, inc) < 1e-12
    assert relerr(naive, inc) > 1e-2
    # with identical a and b parameter sets the naive form holds too
    q = dict(p)
    q["w_b"], q["w_b_gate"], q["b_b"], q["b_b_gate"] = p["w_a"], p["w_a_gate"], p["b_a"], p["b_a_gate"]
    assert relerr(np.transpose(orc.trimul(zT, MT, q, OUT), (1, 0, 2)), orc.trimul(z, M, q, INC)) < 1e-12


@pytest.mark.parametrize("direction", [OUT, INC])
def test_I2_token_permutation_equivariance(direction):
    rng = np.random.default_rng(5)
    N, c_z, c = 7, 8, 4
    z = rng.standard_normal((N, N, c_z))
    m = (rng.random(N) > 0.25).astype(np.float64)
    M = np.outer(m, m)
    p = rand_params(rng, c_z, c)
    pi = rng.permutation(N)
    lhs = orc.trimul(z[pi][:, pi], M[pi][:, pi], p, direction)
    rhs = orc.trimul(z, M, p, direction)[pi][:, pi]
    assert relerr(lhs, rhs) < 1e-12


@pytest.mark.parametrize("direction", [OUT, INC])
def test_I3_masked_tokens_contribute_nothing(direction):
    """Zero contribution from masked tokens: garbage (large, finite) under the mask leaves out
    bitwise unchanged everywhere (mask_output) / on valid pairs (no output mask)."""
    rng = np.random.default_rng(6)
    N, c_z, c = 8, 8, 6
    z = rng.standard_normal((N, N, c_z))
    m = np.ones(N)
    m[[2, 5]] = 0.0
    M = np.outer(m, m)
    p = rand_params(rng, c_z, c)
    z2 = z.copy()
    z2[M == 0] = 100.0 * rng.standard_normal((int((M == 0).sum()), c_z))
    assert np.array_equal(orc.trimul(z, M, p, direction), orc.trimul(z2, M, p, direction))
    o1 = orc.trimul(z, M, p, direction, mask_output=False)
    o2 = orc.trimul(z2, M, p, direction, mask_output=False)
    assert np.array_equal(o1[M == 1], o2[M == 1])
    # and the masked output is exactly zero on masked pairs, non-zero without the output mask (A8/A20)
    assert np.all(orc.trimul(z, M, p, direction)[M == 0] == 0.0)
    assert np.all(np.abs(o1[M == 0]).max(axis=-1) > 0)
    # removing masked tokens altogether gives the same values on the kept block
    keep = np.where(m == 1)[0]
    small = orc.trimul(z[keep][:, keep], None, p, direction)
    assert relerr(small, orc.trimul(z, M, p, direction)[keep][:, keep]) < 1e-12


def test_I6_input_layernorm_shift_and_scale():
    rng = np.random.default_rng(9)
    N, c_z, c = 5, 8, 4
    z = rng.standard_normal((N, N, c_z))
    p = rand_params(rng, c_z, c)
    ref = orc.trimul(z, None, p, OUT)
    shift = rng.standard_normal((N, N, 1))
    assert relerr(orc.trimul(z + shift, None, p, OUT), ref) < 1e-12
    # scaling by s changes out only through eps: with eps=0 exactly invariant, with 1e-5 nearly
    assert relerr(orc.trimul(3.0 * z, None, p, OUT, eps=0.0), orc.trimul(z, None, p, OUT, eps=0.0)) < 1e-12
    assert relerr(orc.trimul(3.0 * z, None, p, OUT), ref) < 1e-4


def test_layer_norm_biased_variance_and_eps_inside_sqrt():
    x = np.array([[1.0, 2.0, 3.0, 6.0]])
    g = np.array([1.0, 2.0, 1.0, 1.0])
    b = np.array([0.0, 0.5, 0.0, 0.0])
    mu, var = 3.0, (4 + 1 + 0 + 9) / 4.0          # biased: 3.5 (unbiased would be 14/3)
    want = (x - mu) / math.sqrt(var + 0.25) * g + b
    assert np.allclose(orc.layer_norm(x, g, b, 0.25), want, rtol=1e-15)
    # degenerate constant row -> beta (A20), finite thanks to eps
    assert np.allclose(orc.layer_norm(np.full((1, 4), 7.0), g, b, 1e-5), b)


def test_sigmoid_values_and_stability():
    assert orc.sigmoid(np.array(0.0)) == 0.5
    assert np.isclose(orc.sigmoid(np.array(math.log(3.0))), 0.75, rtol=1e-15)
    assert np.isclose(orc.sigmoid(np.array(-math.log(3.0))), 0.25, rtol=1e-15)
    with np.errstate(over="raise"):
        v = orc.sigmoid(np.array([-800.0, 800.0]))
    assert v[0] >= 0 and v[0] < 1e-300 and v[1] == 1.0


# ----------------------------------------------------------------------------------------
# closed forms
# ----------------------------------------------------------------------------------------
def _one_pair(zv, p, eps=1e-5):
    """Hand computation for a single feature vector (used by S1)."""
    mu = zv.mean()
    var = ((zv - mu) ** 2).mean()
    zp = (zv - mu) / math.sqrt(var + eps) * p["ln_in_gamma"] + p["ln_in_beta"]
    sg = lambda x: 1 / (1 + np.exp(-x))
    alpha = sg(p["w_a_gate"] @ zp + p["b_a_gate"]) * (p["w_a"] @ zp + p["b_a"])
    beta = sg(p["w_b_gate"] @ zp + p["b_b_gate"]) * (p["w_b"] @ zp + p["b_b"])
    g = sg(p["w_g"] @ zp + p["b_g"])
    return alpha, beta, g


@pytest.mark.parametrize("direction", [OUT, INC])
def test_S1_constant_z(direction):
    rng = np.random.default_rng(10)
    N, c_z, c = 6, 8, 5
    zv = rng.standard_normal(c_z)
    z = np.broadcast_to(zv, (N, N, c_z)).copy()
    p = rand_params(rng, c_z, c)
    alpha, beta, g = _one_pair(zv, p)
    o = N * alpha * beta
    mu, var = o.mean(), ((o - o.mean()) ** 2).mean()
    on = (o - mu) / math.sqrt(var + 1e-5) * p["ln_out_gamma"] + p["ln_out_beta"]
    want = g * (p["w_o"] @ on + p["b_o"])
    got = orc.trimul(z, None, p, direction)
    assert np.allclose(got, np.broadcast_to(want, got.shape), rtol=1e-12, atol=1e-13)


@pytest.mark.parametrize("direction", [OUT, INC])
def test_S2_zero_weights_token_mask(direction):
    """All six W = 0, biases != 0, token mask m: o_ij = m_i m_j (sum_k m_k) alpha*beta."""
    rng = np.random.default_rng(11)
    N, c_z, c = 7, 8, 4
    z = rng.standard_normal((N, N, c_z))
    p = rand_params(rng, c_z, c)
    for k in ("w_a", "w_a_gate", "w_b", "w_b_gate", "w_g"):
        p[k] = np.zeros_like(p[k])
    m = np.array([1, 1, 0, 1, 0, 1, 1.0])
    M = np.outer(m, m)
    sg = lambda x: 1 / (1 + np.exp(-x))
    alpha = sg(p["b_a_gate"]) * p["b_a"]
    beta = sg(p["b_b_gate"]) * p["b_b"]
    g = sg(p["b_g"])
    want = np.zeros((N, N, c_z))
    for i in range(N):
        for j in range(N):
            o = m[i] * m[j] * m.sum() * alpha * beta
            mu, var = o.mean(), ((o - o.mean()) ** 2).mean()
            on = (o - mu) / math.sqrt(var + 1e-5) * p["ln_out_gamma"] + p["ln_out_beta"]
            want[i, j] = M[i, j] * g * (p["w_o"] @ on + p["b_o"])
    assert np.allclose(orc.trimul(z, M, p, direction), want, rtol=1e-12, atol=1e-14)


def test_S3_S4_output_stage_isolated():
    rng = np.random.default_rng(12)
    N, c_z, c = 5, 8, 6
    z = rng.standard_normal((N, N, c_z))
    M = (rng.random((N, N)) > 0.3).astype(np.float64)
    p = rand_params(rng, c_z, c)
    # S3: gamma_out = 0 -> out_ij = M_ij g_ij * (W_o beta_out + b_o), independent of the contraction
    q = dict(p)
    q["ln_out_gamma"] = np.zeros(c)
    zp = orc.layer_norm(z, p["ln_in_gamma"], p["ln_in_beta"], 1e-5)
    g = 1 / (1 + np.exp(-(zp @ p["w_g"].T + p["b_g"])))
    want = M[..., None] * g * (p["w_o"] @ p["ln_out_beta"] + p["b_o"])
    for d in (OUT, INC):
        assert np.allclose(orc.trimul(z, M, q, d), want, rtol=1e-12, atol=1e-14)
    # S4: W_o = 0, b_o = 0 -> out == 0 exactly
    q = dict(p)
    q["w_o"] = np.zeros_like(p["w_o"])
    q["b_o"] = np.zeros(c_z)
    assert np.all(orc.trimul(z, M, q, OUT) == 0.0)


def test_S8_symmetric_input_directions_coincide():
    rng = np.random.default_rng(13)
    N, c_z, c = 6, 8, 5
    z = rng.standard_normal((N, N, c_z))
    z = z + np.transpose(z, (1, 0, 2))
    m = (rng.random(N) > 0.2).astype(np.float64)
    M = np.outer(m, m)
    p = rand_params(rng, c_z, c)
    assert relerr(orc.trimul(z, M, p, OUT), orc.trimul(z, M, p, INC)) < 1e-13


def test_N1_single_token():
    rng = np.random.default_rng(14)
    c_z, c = 8, 4
    zv = rng.standard_normal(c_z)
    p = rand_params(rng, c_z, c)
    alpha, beta, g = _one_pair(zv, p)
    o = alpha * beta
    mu, var = o.mean(), ((o - o.mean()) ** 2).mean()
    on = (o - mu) / math.sqrt(var + 1e-5) * p["ln_out_gamma"] + p["ln_out_beta"]
    want = g * (p["w_o"] @ on + p["b_o"])
    for d in (OUT, INC):
        assert np.allclose(orc.trimul(zv[None, None], None, p, d)[0, 0], want, rtol=1e-12)


def test_output_ln_scale_invariance_loose():
    rng = np.random.default_rng(15)
    N, c_z, c = 6, 8, 5
    z = rng.standard_normal((N, N, c_z))
    p = rand_params(rng, c_z, c)
    ref = orc.trimul(z, None, p, OUT)
    for s in (0.5, 2.0):
        q = dict(p)
        q["w_a"], q["b_a"] = s * p["w_a"], s * p["b_a"]
        assert relerr(orc.trimul(z, None, q, OUT), ref) < 1e-4


# ----------------------------------------------------------------------------------------
# sub-grid oracle == full oracle on the sampled pairs
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("direction", [OUT, INC])
@pytest.mark.parametrize("mask_output", [True, False])
def test_subgrid_matches_full(direction, mask_output):
    rng = np.random.default_rng(16)
    N, c_z, c = 11, 8, 6
    z = rng.standard_normal((N, N, c_z))
    M = (rng.random((N, N)) > 0.3).astype(np.float64)
    p = rand_params(rng, c_z, c)
    I = np.array([0, 3, 10, 4])
    J = np.array([10, 1, 2])
    if direction == OUT:
        za, ma, zb, mb = z[I], M[I], z[J], M[J]
    else:
        za, ma = np.transpose(z[:, I], (1, 0, 2)), M[:, I].T
        zb, mb = np.transpose(z[:, J], (1, 0, 2)), M[:, J].T
    got = orc.trimul_subgrid(za, ma, zb, mb, z[I][:, J], M[I][:, J], p, mask_output=mask_output)
    full = orc.trimul(z, M, p, direction, mask_output=mask_output)
    assert relerr(got, full[I][:, J]) < 1e-12


# ----------------------------------------------------------------------------------------
# row-block form (bounded memory, used for whole-tensor parity at N = 4096): pinned against the
# scalar loops and against the whole-tensor oracle, both directions, general pair mask, ragged
# blocks, projections evaluated slice by slice
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("direction", [OUT, INC])
@pytest.mark.parametrize("mask_output", [True, False])
def test_rowblock_against_brute_force_and_full(direction, mask_output):
    rng = np.random.default_rng(77 + direction)
    N, c_z, c = 7, 8, 5
    z = rng.standard_normal((N, N, c_z))
    M = (rng.random((N, N)) > 0.3).astype(np.float64)       # general, non-symmetric pair mask
    p = rand_params(rng, c_z, c)
    # projections of the whole z, evaluated in row slices of unequal height
    a = np.empty((N, N, c))
    b = np.empty((N, N, c))
    for r0, r1 in ((0, 2), (2, 3), (3, 7)):
        a[r0:r1], b[r0:r1] = orc.projections(z[r0:r1], M[r0:r1], p)
    blocks = [(0, 3), (3, 4), (4, 7)]                         # ragged row blocks
    got = np.concatenate([orc.trimul_rowblock(a, b, z[i0:i1], M[i0:i1], p, direction, i0, i1,
                                              mask_output=mask_output) for i0, i1 in blocks])
    brute = np.array(brute_force.trimul_brute(z.tolist(), M.tolist(), tolist(p), direction,
                                              mask_output=mask_output))
    assert got.shape == (N, N, c_z)
    assert relerr(got, brute) < 1e-12
    assert relerr(got, orc.trimul(z, M, p, direction, mask_output=mask_output)) < 1e-13
    # a transposed operand or a swapped direction must not pass: the two directions differ
    other = np.concatenate([orc.trimul_rowblock(a, b, z[i0:i1], M[i0:i1], p, 1 - direction, i0, i1,
                                                mask_output=mask_output) for i0, i1 in blocks])
    assert relerr(other, brute) > 1e-2


def test_rowblock_null_mask_and_single_row():
    rng = np.random.default_rng(5)
    N, c_z, c = 5, 4, 6
    z = rng.standard_normal((N, N, c_z))
    p = rand_params(rng, c_z, c, bias=False)
    a, b = orc.projections(z, None, p)
    for direction in (OUT, INC):
        full = orc.trimul(z, None, p, direction)
        for i in range(N):
            row = orc.trimul_rowblock(a, b, z[i:i + 1], None, p, direction, i, i + 1)
            assert relerr(row[0], full[i]) < 1e-13


# ----------------------------------------------------------------------------------------
# backward pass: finite differences of the forward
# oracle for every input and parameter, the adjoint identity, scalar-loop LayerNorm Jacobian
# ----------------------------------------------------------------------------------------
def _fd(f, x, idx, h=1e-6):
    """central difference of the scalar function f with respect to x[idx]"""
    old = x[idx]
    x[idx] = old + h
    fp = f()
    x[idx] = old - h
    fm = f()
    x[idx] = old
    return (fp - fm) / (2 * h)


@pytest.mark.parametrize("direction", [OUT, INC])
@pytest.mark.parametrize("mask_output,bias", [(True, True), (False, False)])
def test_backward_against_finite_differences(direction, mask_output, bias):
    rng = np.random.default_rng(900 + 10 * direction + int(bias))
    N, c_z, c = 4, 6, 5
    z = rng.standard_normal((N, N, c_z))
    M = (rng.random((N, N)) > 0.25).astype(np.float64)
    M[1, 2] = 0.5                                               # a soft mask value too (A22)
    p = rand_params(rng, c_z, c, bias=bias)
    d_out = rng.standard_normal((N, N, c_z))
    loss = lambda: float((d_out * orc.trimul(z, M, p, direction, mask_output=mask_output)).sum())
    d_z, grads = orc.trimul_backward(d_out, z, M, p, direction, mask_output=mask_output)
    assert set(grads) == set(p)                                 # every parameter has a gradient
    # d_z: every element
    for idx in np.ndindex(z.shape):
        assert abs(_fd(loss, z, idx) - d_z[idx]) < 2e-7 * max(1.0, abs(d_z[idx])), ("z", idx)
    # parameters: every element of the vectors, a seeded sample of the matrices
    for name, arr in p.items():
        gr = grads[name]
        assert gr.shape == arr.shape, name
        idxs = list(np.ndindex(arr.shape))
        if arr.ndim == 2:
            idxs = [idxs[k] for k in rng.choice(len(idxs), size=12, replace=False)]
        for idx in idxs:
            assert abs(_fd(loss, arr, idx) - gr[idx]) < 2e-7 * max(1.0, abs(gr[idx])), (name, idx)


@pytest.mark.parametrize("direction", [OUT, INC])
def test_backward_adjoint_identity_and_residual(direction):
    """<d_out, J u> = <J^T d_out, u> with J u from a central difference along a random direction u
    of ALL inputs at once (z and every parameter); the residual form adds d_out to d_z."""
    rng = np.random.default_rng(77 + direction)
    N, c_z, c = 6, 8, 4
    z = rng.standard_normal((N, N, c_z))
    M = (rng.random((N, N)) > 0.3).astype(np.float64)
    p = rand_params(rng, c_z, c)
    d_out = rng.standard_normal((N, N, c_z))
    uz = rng.standard_normal(z.shape)
    up = {k: rng.standard_normal(v.shape) for k, v in p.items()}
    h = 1e-6
    shift = lambda t: (z + t * uz, {k: v + t * up[k] for k, v in p.items()})
    zp_, pp_ = shift(h)
    zm_, pm_ = shift(-h)
    Ju = (orc.trimul(zp_, M, pp_, direction) - orc.trimul(zm_, M, pm_, direction)) / (2 * h)
    d_z, grads = orc.trimul_backward(d_out, z, M, p, direction)
    lhs = float((d_out * Ju).sum())
    rhs = float((d_z * uz).sum()) + sum(float((grads[k] * up[k]).sum()) for k in p)
    assert abs(lhs - rhs) < 1e-6 * max(1.0, abs(lhs))
    d_z_res, grads_res = orc.trimul_backward(d_out, z, M, p, direction, residual=True)
    assert np.array_equal(d_z_res, d_z + d_out)
    assert all(np.array_equal(grads_res[k], grads[k]) for k in grads)


def test_layer_norm_backward_against_scalar_jacobian():
    """d_x of the LayerNorm from its Jacobian written out element by element in Python floats:
    dy_t/dx_s = gamma_t * rstd * (delta_ts - 1/n - xh_t xh_s / n)."""
    rng = np.random.default_rng(3)
    n, eps = 7, 1e-3
    x = rng.standard_normal(n).tolist()
    gamma = (1 + 0.3 * rng.standard_normal(n)).tolist()
    dy = rng.standard_normal(n).tolist()
    mu = sum(x) / n
    var = sum((v - mu) ** 2 for v in x) / n
    rstd = 1.0 / math.sqrt(var + eps)
    xh = [(v - mu) * rstd for v in x]
    dx = [sum(dy[t] * gamma[t] * rstd * ((1.0 if t == s_ else 0.0) - 1.0 / n - xh[t] * xh[s_] / n)
              for t in range(n)) for s_ in range(n)]
    got_dx, got_dg, got_db = orc.layer_norm_backward(np.array([dy]), np.array([x]), np.array(gamma), eps)
    assert np.allclose(got_dx[0], dx, rtol=0, atol=1e-13)
    assert np.allclose(got_dg, [dy[t] * xh[t] for t in range(n)], rtol=0, atol=1e-13)
    assert np.allclose(got_db, dy, rtol=0, atol=1e-15)


# ----------------------------------------------------------------------------------------
# the paper's Cannon-style distributed contraction, simulated grid
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("grid", [1, 2, 3, 4])
@pytest.mark.parametrize("direction", [OUT, INC])
def test_cannon_contraction_equals_definition(grid, direction):
    rng = np.random.default_rng(50 + grid)
    N, c = 12, 3
    a = rng.standard_normal((N, N, c))
    b = rng.standard_normal((N, N, c))
    got = orc.contraction_cannon(a, b, direction, grid)
    # against the scalar definition of Eq. 2-3 written out here, not against orc.contraction
    ref = np.zeros((N, N, c))
    for i in range(N):
        for j in range(N):
            for k in range(N):
                ref[i, j] += (a[i, k] * b[j, k]) if direction == OUT else (a[k, i] * b[k, j])
    assert relerr(got, ref) < 1e-13


@pytest.mark.parametrize("grid", [2, 3, 4])
@pytest.mark.parametrize("direction", [OUT, INC])
def test_cannon_schedule_is_a_ring(grid, direction):
    """Every rank meets every contracted block index exactly once; between consecutive steps the a
    block it needs is the one its right-hand neighbour (r, c+1) just used and the b block the one
    its lower neighbour (r+1, c) just used: one nearest-neighbour shift along rows / columns per
    step, as PAPER.md lines 132-134 describe."""
    sched = orc.cannon_schedule(grid, direction)
    for (r, c), steps in sched.items():
        qs = [(ab[0][1] if direction == OUT else ab[0][0]) for ab in steps]
        assert sorted(qs) == list(range(grid))
        for s_ in range(grid):
            ablk, bblk = steps[s_]
            # the two blocks share the contracted block index, and they are the blocks the
            # definition pairs: a_(r,q) b_(c,q) (outgoing), a_(q,r) b_(q,c) (incoming)
            if direction == OUT:
                assert ablk[0] == r and bblk[0] == c and ablk[1] == bblk[1]
            else:
                assert ablk[1] == r and bblk[1] == c and ablk[0] == bblk[0]
            if s_ + 1 < grid:
                assert sched[(r, (c + 1) % grid)][s_][0] == steps[s_ + 1][0]      # a arrives from the right
                assert sched[((r + 1) % grid, c)][s_][1] == steps[s_ + 1][1]      # b arrives from below


@pytest.mark.parametrize("direction", [OUT, INC])
def test_trimul_cannon_equals_serial_op(direction):
    """The paper's own validation: the distributed result equals the serial one (lines 23, 221)."""
    rng = np.random.default_rng(8 + direction)
    N, c_z, c = 6, 8, 5
    z = rng.standard_normal((N, N, c_z))
    M = (rng.random((N, N)) > 0.3).astype(np.float64)
    p = rand_params(rng, c_z, c)
    for grid in (2, 3):
        assert relerr(orc.trimul_cannon(z, M, p, direction, grid), orc.trimul(z, M, p, direction)) < 1e-13
    with pytest.raises(ValueError):
        orc.contraction_cannon(np.zeros((5, 5, 1)), np.zeros((5, 5, 1)), direction, 2)


def test_flop_count_matches_baseline_md():
    # 17.592 + 2.749 + 0.550 = 20.891 TFLOP at N=4096, c=c_z=128
    assert abs(orc.flops(4096, 128, 128) / 1e12 - 20.891) < 1e-3
    assert abs(orc.flops(64, 128, 128) / 1e9 - 0.872) < 1e-3


def test_golden_worked_example():
    """Stored tiny worked example (written by tests/golden/make_trimul_golden.py from the scalar
    brute force; the paper prints no numerical example of its own)."""
    import json
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "trimul_n3.json")
    with open(path) as f:
        doc = json.load(f)
    p = {k: np.array(v) for k, v in doc["params"].items()}
    z, M = np.array(doc["z"]), np.array(doc["mask"])
    for d in (OUT, INC):
        for mo in (True, False):
            want = np.array(doc["out"][f"dir{d}_maskout{int(mo)}"])
            got = orc.trimul(z, M, p, d, eps=doc["eps"], mask_output=mo)
            assert np.allclose(got, want, rtol=1e-12, atol=1e-14)
