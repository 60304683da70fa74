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
    e["outputs"] = int(np.asarray(ref).size)
    record_parity(what, e, dtype)      # recorded before asserting: a failing run leaves its numbers
    assert np.all(np.isfinite(np.asarray(got, np.float64))), f"{what}: non-finite output"
    assert e["rel_fro"] <= tol["rel_fro"], f"{what}: rel Frobenius {e['rel_fro']:.3e} > {tol['rel_fro']}"
    assert e["max_over_rms"] <= tol["max_over_rms"], \
        f"{what}: max abs / rms {e['max_over_rms']:.3e} > {tol['max_over_rms']}"
    return e


# ------------------------------------------------------------------------------------------------
# measured-error records: every parity test prints what it measured and appends it to a JSON-lines
# file (gpurun_out/ is the only folder that comes back from the GPU box); tests/parity_report.py
# turns those lines into the tracked profiles/parity_r*.json
# ------------------------------------------------------------------------------------------------
import json
import os
import time

_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def record_parity(what, e, dtype, **fields):
    tol = TOL[dtype]
    rec = dict(what=what, dtype=dtype, rel_fro=e["rel_fro"], max_over_rms=e["max_over_rms"],
               rms=e.get("rms"), tol_rel_fro=tol["rel_fro"], tol_max_over_rms=tol["max_over_rms"],
               margin_rel_fro=1.0 - e["rel_fro"] / tol["rel_fro"],
               margin_max_over_rms=1.0 - e["max_over_rms"] / tol["max_over_rms"],
               when=time.strftime("%Y-%m-%dT%H:%M:%SZ", time.gmtime()))
    for k in ("outputs", "argmax", "max_abs"):
        if k in e:
            rec[k] = e[k]
    rec.update(fields)
    print(f"[parity] {what}: rel_fro={e['rel_fro']:.3e} (tol {tol['rel_fro']:.0e}) "
          f"max/rms={e['max_over_rms']:.3e} (tol {tol['max_over_rms']:.0e})", flush=True)
    path = os.environ.get("FOLDCP_PARITY_LOG", os.path.join(_ROOT, "gpurun_out", "parity_records.jsonl"))
    try:
        os.makedirs(os.path.dirname(path), exist_ok=True)
        with open(path, "a") as f:
            f.write(json.dumps(rec) + "\n")
    except OSError:
        pass
    return rec


# ------------------------------------------------------------------------------------------------
# whole-tensor oracle walk (N = 4096: out alone is 17 GB in fp64): the projections a, b of the
# whole z are evaluated slice by slice (orc.projections), then orc.trimul_rowblock gives the exact
# out[i0:i1] block by block and the error sums are accumulated.  The arithmetic is the oracle's;
# this harness only slices, runs blocks on host threads and adds up squared errors.
# ------------------------------------------------------------------------------------------------
def _host_workers(bytes_per_worker):
    import psutil
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    avail = psutil.virtual_memory().available
    return max(1, min(cores, int(0.6 * avail // max(bytes_per_worker, 1))))


def _projections_cm(z_sel, M_sel, p, keep, eps=1e-5, chunk_rows=16):
    """orc.projections over a [R1, R2, c_z] selection of z (device or host tensor), slice by slice on
    host threads; returns the kept tensors ("a", "b" or "ab") as fp64 [R1, R2, c] views over
    channel-major storage (the layout in which trimul_rowblock's per-channel matmuls read contiguous
    matrices)."""
    from concurrent.futures import ThreadPoolExecutor
    from threadpoolctl import threadpool_limits
    R1, R2, c_z = z_sel.shape
    q = params64(p)
    c = q["w_a"].shape[0]
    store = {k: np.empty((c, R1, R2), np.float64) for k in keep}

    def work(r0):
        r1 = min(R1, r0 + chunk_rows)
        zc = np64(z_sel[r0:r1]).reshape(-1, c_z)
        mc = None if M_sel is None else np64(M_sel[r0:r1]).reshape(-1)
        a, b = orc.projections(zc, mc, q, eps)
        for k, v in (("a", a), ("b", b)):
            if k in store:
                store[k][:, r0:r1, :] = v.reshape(r1 - r0, R2, c).transpose(2, 0, 1)

    workers = _host_workers(chunk_rows * R2 * c_z * 8 * 12)
    with threadpool_limits(limits=1):
        with ThreadPoolExecutor(workers) as ex:
            list(ex.map(work, range(0, R1, chunk_rows)))
    return tuple(store[k].transpose(1, 2, 0) for k in keep)


def oracle_projections_whole(z, M, p, eps=1e-5, chunk_rows=16):
    """(a, b) of the whole z as fp64 [N, N, c] views (channel-major storage)."""
    return _projections_cm(z, M, p, "ab", eps, chunk_rows)


def whole_tensor_errors(out, z, M, p, direction, row_blocks=None, block_rows=32, mask_output=True,
                        eps=1e-5, ab=None, rows=None):
    """Errors of `out` (device or host tensor [N, N, c_z]) against the oracle over the given row
    blocks (default: every row, i.e. the WHOLE tensor).  Returns rel_fro, max_over_rms (rms over the
    compared oracle outputs), the arg-max location and the number of outputs compared.

    rows = sorted index array: only those output rows are compared (all columns).  Then b is
    evaluated for the whole z but a only where Eq. 2-3 need it -- rows `rows` (outgoing) or columns
    `rows` (incoming) -- and handed to trimul_rowblock in compacted form (N = 8192: a and b whole
    would be 137 GB in fp64)."""
    from concurrent.futures import ThreadPoolExecutor
    from threadpoolctl import threadpool_limits
    import torch
    N, c_z = z.shape[0], z.shape[2]
    q = params64(p)
    c = q["w_a"].shape[0]
    if rows is not None:
        rows = np.asarray(rows, dtype=np.int64)
        rt = torch.as_tensor(rows, device=z.device)
        (b,) = _projections_cm(z, M, p, "b", eps)
        if direction == orc.OUTGOING:
            (a,) = _projections_cm(z[rt], None if M is None else M[rt], p, "a", eps)
        else:
            (a,) = _projections_cm(z[:, rt], None if M is None else M[:, rt], p, "a", eps)
        nsel = rows.size
        if row_blocks is None:
            row_blocks = [(i0, min(nsel, i0 + block_rows)) for i0 in range(0, nsel, block_rows)]
        sel = lambda t, i0, i1: t[torch.as_tensor(rows[i0:i1], device=t.device)]
        row_of = lambda i: int(rows[i])
    else:
        a, b = ab if ab is not None else oracle_projections_whole(z, M, p, eps)
        if row_blocks is None:
            row_blocks = [(i0, min(N, i0 + block_rows)) for i0 in range(0, N, block_rows)]
        sel = lambda t, i0, i1: t[i0:i1]
        row_of = lambda i: i

    def work(blk):
        i0, i1 = blk
        ref = orc.trimul_rowblock(a, b, np64(sel(z, i0, i1)), None if M is None else np64(sel(M, i0, i1)),
                                  q, direction, i0, i1, eps=eps, mask_output=mask_output)
        got = np64(sel(out, i0, i1))
        d = np.abs(got - ref)
        k = int(np.argmax(d))
        return (float((d * d).sum()), float((ref * ref).sum()), float(d.flat[k]),
                tuple(int(v) for v in np.unravel_index(k, d.shape)), i0, ref.size,
                bool(np.all(np.isfinite(got))))

    workers = _host_workers(block_rows * N * max(c, c_z) * 8 * 12)
    with threadpool_limits(limits=1):
        with ThreadPoolExecutor(workers) as ex:
            res = list(ex.map(work, row_blocks))
    sd = sum(r[0] for r in res)
    sr = sum(r[1] for r in res)
    n = sum(r[5] for r in res)
    worst = max(res, key=lambda r: r[2])
    rms = (sr / n) ** 0.5
    return dict(rel_fro=(sd / max(sr, 1e-300)) ** 0.5, max_over_rms=worst[2] / max(rms, 1e-300),
                rms=rms, max_abs=worst[2], argmax=[row_of(worst[4] + worst[3][0]), worst[3][1], worst[3][2]],
                outputs=n, finite=all(r[6] for r in res), host_workers=workers)
