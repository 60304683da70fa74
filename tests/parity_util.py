"""Helpers for the GPU-vs-oracle parity tests: oracle evaluation (full or sub-grid) from the very
tensors handed to the library, error metrics, and BASELINE.json's tolerances."""
import numpy as np
import torch

from oracle import trimul_oracle as orc

# BASELINE.json north_star: bf16 -> relative Frobenius <= 1e-2 and max abs <= 5e-2 * rms(out);
# fp32 mode -> relative error <= 1e-5 (reading A11: relative Frobenius)
TOL = {"bf16": dict(rel_fro=1e-2, max_over_rms=5e-2), "f32": dict(rel_fro=1e-5, max_over_rms=1e-4)}


def np64(t):
    return t.detach().to("cpu", torch.float64).numpy()


def params64(p):
    return {k: (None if v is None else np64(v)) for k, v in p.items()}


def oracle_full(z, M, p, direction, mask_output=True, eps=1e-5):
    return orc.trimul(np64(z), None if M is None else np64(M), params64(p), direction, eps=eps,
                      mask_output=mask_output)


def oracle_subgrid(z, M, p, direction, I, J, mask_output=True, eps=1e-5):
    """Exact out[I x J]; pulls only the needed rows / columns of z (which may live on the GPU)."""
    It = torch.as_tensor(I, device=z.device)
    Jt = torch.as_tensor(J, device=z.device)
    if direction == orc.OUTGOING:
        za, zb = z[It], z[Jt]
        ma = mb = None
        if M is not None:
            ma, mb = M[It], M[Jt]
    else:
        za, zb = z[:, It].transpose(0, 1), z[:, Jt].transpose(0, 1)
        ma = mb = None
        if M is not None:
            ma, mb = M[:, It].t(), M[:, Jt].t()
    zij = z[It][:, Jt]
    mij = None if M is None else M[It][:, Jt]
    f = lambda t: None if t is None else np64(t.contiguous())
    return orc.trimul_subgrid(f(za), f(ma), f(zb), f(mb), f(zij), f(mij), params64(p), eps=eps,
                              mask_output=mask_output)


def sample_indices(N, n, seed, tile=128, extra=()):
    """Index set that hits both sides of every `tile` boundary it can afford, the first / last
    index, `extra` (e.g. masked tokens) and seeded random picks -- n indices in all."""
    rng = np.random.default_rng(seed)
    must = {0, N - 1}
    for b in range(tile, N, tile):
        must.update((b - 1, b))
    must.update(int(e) for e in extra)
    must = sorted(must)
    if len(must) > n:
        must = sorted(rng.choice(must, size=n, replace=False).tolist() + [0, N - 1])[:n]
    rest = np.setdiff1d(np.arange(N), np.array(must))
    more = rng.choice(rest, size=max(0, n - len(must)), replace=False)
    return np.sort(np.concatenate([np.array(must, dtype=np.int64), more.astype(np.int64)]))


def errors(got, ref):
    got = np.asarray(got, np.float64)
    d = got - ref
    rms = np.sqrt(np.mean(ref ** 2))
    return dict(rel_fro=float(np.linalg.norm(d) / max(np.linalg.norm(ref), 1e-300)),
                max_over_rms=float(np.abs(d).max() / max(rms, 1e-300)), rms=float(rms))


def assert_parity(got, ref, dtype, what=""):
    e = errors(got, ref)
    tol = TOL[dtype]
    assert np.all(np.isfinite(np.asarray(got, np.float64))), f"{what}: non-finite output"
    assert e["rel_fro"] <= tol["rel_fro"], f"{what}: rel Frobenius {e['rel_fro']:.3e} > {tol['rel_fro']}"
    assert e["max_over_rms"] <= tol["max_over_rms"], \
        f"{what}: max abs / rms {e['max_over_rms']:.3e} > {tol['max_over_rms']}"
    return e
