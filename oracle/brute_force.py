"""Index-by-index restatement of the triangle multiplicative update in pure Python floats.

TEST INFRASTRUCTURE.  A deliberately naive second implementation (scalar loops, `math` only,
no numpy, no shared helpers) used ONLY to pin oracle/trimul_oracle.py on tiny shapes
(tests/test_oracle_pins.py).  Follows PAPER.md Eq. 2-3 (lines 121-128) and the north_star
statement of the op literally, one scalar at a time.
"""
import math

OUTGOING = 0
INCOMING = 1


def _sigmoid(x):
    if x >= 0.0:
        return 1.0 / (1.0 + math.exp(-x))
    e = math.exp(x)
    return e / (1.0 + e)


def _layer_norm_vec(v, gamma, beta, eps):
    n = len(v)
    mu = sum(v) / n
    var = sum((x - mu) * (x - mu) for x in v) / n
    r = 1.0 / math.sqrt(var + eps)
    return [(v[t] - mu) * r * gamma[t] + beta[t] for t in range(n)]


def _matvec(w, x, b):
    out = []
    for r in range(len(w)):
        s = 0.0
        for t in range(len(x)):
            s += w[r][t] * x[t]
        out.append(s + (b[r] if b is not None else 0.0))
    return out


def trimul_brute(z, mask, p, direction, eps=1e-5, mask_output=True):
    """z: nested lists [N][N][c_z]; mask: [N][N] or None; p: dict of nested lists.
    Returns nested lists [N][N][c_z]."""
    N = len(z)
    c = len(p["w_a"])
    c_z = len(p["w_g"])
    zp = [[_layer_norm_vec(z[i][j], p["ln_in_gamma"], p["ln_in_beta"], eps)
           for j in range(N)] for i in range(N)]
    a = [[None] * N for _ in range(N)]
    b = [[None] * N for _ in range(N)]
    g = [[None] * N for _ in range(N)]
    for i in range(N):
        for j in range(N):
            m = 1.0 if mask is None else mask[i][j]
            pa = _matvec(p["w_a"], zp[i][j], p.get("b_a"))
            ga = _matvec(p["w_a_gate"], zp[i][j], p.get("b_a_gate"))
            pb = _matvec(p["w_b"], zp[i][j], p.get("b_b"))
            gb = _matvec(p["w_b_gate"], zp[i][j], p.get("b_b_gate"))
            a[i][j] = [m * _sigmoid(ga[t]) * pa[t] for t in range(c)]
            b[i][j] = [m * _sigmoid(gb[t]) * pb[t] for t in range(c)]
            g[i][j] = [_sigmoid(x) for x in _matvec(p["w_g"], zp[i][j], p.get("b_g"))]
    out = [[None] * N for _ in range(N)]
    for i in range(N):
        for j in range(N):
            o = [0.0] * c
            for k in range(N):
                for t in range(c):
                    if direction == OUTGOING:
                        o[t] += a[i][k][t] * b[j][k][t]      # Eq. 2
                    else:
                        o[t] += a[k][i][t] * b[k][j][t]      # Eq. 3
            on = _layer_norm_vec(o, p["ln_out_gamma"], p["ln_out_beta"], eps)
            y = _matvec(p["w_o"], on, p.get("b_o"))
            m = 1.0 if (mask is None or not mask_output) else mask[i][j]
            out[i][j] = [m * g[i][j][t] * y[t] for t in range(c_z)]
    return out
