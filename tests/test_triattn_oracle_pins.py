"""Pins of oracle/triattn_oracle.py (Eq. 1): brute force on
tiny shapes, invariants and special cases chosen so that a dropped term, a wrong axis or a transposed
operand fails one of them.  CPU only."""
import numpy as np
import pytest

from oracle import triattn_oracle as ta

S, E = ta.STARTING, ta.ENDING


def make(N, cz, H, c, seed, mask_p=0.0):
    r = np.random.default_rng(seed)
    z = r.normal(size=(N, N, cz))
    p = dict(ln_gamma=1 + 0.1 * r.normal(size=cz), ln_beta=0.1 * r.normal(size=cz),
             w_q=r.normal(size=(H * c, cz)) / np.sqrt(cz), w_k=r.normal(size=(H * c, cz)) / np.sqrt(cz),
             w_v=r.normal(size=(H * c, cz)) / np.sqrt(cz), w_g=r.normal(size=(H * c, cz)) / np.sqrt(cz),
             w_t=r.normal(size=(H, cz)) / np.sqrt(cz), w_o=r.normal(size=(cz, H * c)) / np.sqrt(H * c))
    M = None
    if mask_p > 0:
        m = (r.uniform(size=N) > mask_p).astype(np.float64)
        m[0] = 1.0
        M = np.outer(m, m)
        M[:, 0] = 1.0            # general (non outer-product) masks too; every row keeps a key
        M[0, :] = 1.0
    return z, M, p


@pytest.mark.parametrize("node", [S, E])
@pytest.mark.parametrize("N,cz,H,c,mask_p", [(1, 4, 1, 2, 0.0), (2, 4, 2, 2, 0.0), (3, 6, 2, 3, 0.4), (5, 8, 4, 2, 0.3)])
def test_brute_force(node, N, cz, H, c, mask_p):
    z, M, p = make(N, cz, H, c, 10 * N + node, mask_p)
    ref = np.array(ta.triattn_brute(z.tolist(), None if M is None else M.tolist(),
                                    {k: v.tolist() for k, v in p.items()}, node, H))
    got = ta.triangle_attention(z, M, p, node, H)
    assert np.abs(got - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max())


@pytest.mark.parametrize("node", [S, E])
def test_attention_rows_sum_to_one_and_masked_keys_get_zero(node):
    z, M, p = make(6, 8, 2, 4, 3, 0.4)
    q, k, v, g, t = ta.projections(z, p, 2)
    a = ta.attention_weights(q, k, t, M, node)
    assert np.abs(a.sum(axis=2) - 1.0).max() < 1e-13
    key_mask = M[:, None, :] if node == S else M.T[None, :, :]      # mb_ik / mb_kj
    assert np.all(a[np.broadcast_to(key_mask[..., None] == 0, a.shape)] == 0.0)


def test_ending_node_is_the_starting_node_on_the_transposed_input():
    z, M, p = make(5, 8, 2, 4, 7, 0.3)
    e = ta.triangle_attention(z, M, p, E, 2)
    s = ta.triangle_attention(np.transpose(z, (1, 0, 2)), M.T, p, S, 2)
    assert np.abs(e - np.transpose(s, (1, 0, 2))).max() < 1e-12
    # and the two nodes really differ on a non-symmetric input
    assert np.abs(e - ta.triangle_attention(z, M, p, S, 2)).max() > 1e-3


@pytest.mark.parametrize("node", [S, E])
def test_uniform_attention_closed_form(node):
    """W_q = 0 and W_t = 0: every score is 0, the weights are 1/N, o_ij = g_ij * mean_k v."""
    N, H, c = 4, 2, 3
    z, _, p = make(N, 6, H, c, 11)
    p["w_q"] = np.zeros_like(p["w_q"])
    p["w_t"] = np.zeros_like(p["w_t"])
    q, k, v, g, t = ta.projections(z, p, H)
    vm = v.mean(axis=1, keepdims=True) if node == S else v.mean(axis=0, keepdims=True)
    ref = (g * np.broadcast_to(vm, v.shape)).reshape(N, N, -1) @ p["w_o"].T
    assert np.abs(ta.triangle_attention(z, None, p, node, H) - ref).max() < 1e-12


@pytest.mark.parametrize("node", [S, E])
def test_triangular_bias_axis(node):
    """Only the bias term couples j and k (starting) / k and i (ending): with W_q = 0 the weights must be
    softmax over k of t_jk (starting) or t_ki (ending) -- a transposed bias fails this."""
    N, H, c = 5, 2, 2
    z, _, p = make(N, 6, H, c, 13)
    p["w_q"] = np.zeros_like(p["w_q"])
    q, k, v, g, t = ta.projections(z, p, H)
    a = ta.attention_weights(q, k, t, None, node)
    for i in range(N):
        for j in range(N):
            col = t[j, :, :] if node == S else t[:, i, :]
            e = np.exp(col - col.max(axis=0))
            assert np.abs(a[i, j] - e / e.sum(axis=0)).max() < 1e-13


@pytest.mark.parametrize("node", [S, E])
def test_token_permutation_equivariance(node):
    z, M, p = make(6, 8, 2, 4, 17, 0.3)
    pi = np.random.default_rng(5).permutation(6)
    a = ta.triangle_attention(z[pi][:, pi], M[pi][:, pi], p, node, 2)
    b = ta.triangle_attention(z, M, p, node, 2)[pi][:, pi]
    assert np.abs(a - b).max() < 1e-12


def test_flop_count():
    assert ta.flops(4096, 128, 4, 32) == 4.0 * 4096 ** 3 * 128 + 2.0 * 4096 ** 2 * 128 * 516 + 2.0 * 4096 ** 2 * 128 * 128
