#!/usr/bin/env python
"""Benchmark of the triangle multiplicative update hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--n 4096]

A "step" is one pass of the whole hot path over one synthetic pair tensor: the OUTGOING and the
INCOMING triangle multiplicative update (two foldcp_trimul calls, separate parameter sets -- every
BASELINE config is "outgoing+incoming") on z[N, N, 128] bf16, N = 4096 (BASELINE configs[3], the
config the metric is quoted on).  Prints ONE JSON line (rank 0).  Multi-GPU: replicas only (the path
is not sharded -- north_star), one process per GPU, value = all ranks' FLOPs / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

C = 128


def k2_traffic_from_profile():
    """dram__bytes_read.sum + dram__bytes_write.sum of one k2_contract launch at N = 4096, parsed from
    the newest committed ncu --set full summary (profiles/r<round>_k2_contract_ncu_full.txt).
    Returns (bytes or None, file name or None): nothing is hard-coded here."""
    import glob
    import re
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r[0-9]*_k2_contract_ncu_full.txt")),
                   key=lambda f: int(re.match(r"r(\d+)", os.path.basename(f)).group(1)))
    if not files:
        return None, None
    rd = wr = None
    with open(files[-1]) as f:
        for line in f:
            m = re.match(r"dram__bytes_(read|write)\.sum \[(\w+)\]:\s*([0-9.eE+-]+)", line)
            if m:
                unit = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0}[m.group(2)]
                v = float(m.group(3)) * unit
                if m.group(1) == "read":
                    rd = v
                else:
                    wr = v
    if rd is None or wr is None:
        return None, os.path.basename(files[-1])
    return rd + wr, os.path.basename(files[-1])


def counted_flops(N: int) -> float:
    """2cN^3 + 2N^2 c_z(4c + c_z) + 2N^2 c c_z per call."""
    return 2.0 * C * N ** 3 + 2.0 * N * N * C * (4 * C + C) + 2.0 * N * N * C * C


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return dict(hbm_gbs=d["hbm_gbs"], tf_burst=d["bf16_tflops"],
                    tf_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]), source="measured")
    # fallback stated in B200_PROFILING.md
    return dict(hbm_gbs=6650.0, tf_burst=1590.0, tf_sustained=1400.0, source="fallback")


def max_over_ranks(ms: float, world: int, dist=None, device="cpu") -> float:
    """Replicas only: every rank times its own replica; the job's time is the slowest rank's."""
    if world <= 1:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_tflops(flops_per_rank_step: float, ms_per_step: float, world: int) -> float:
    """value = the FLOPs all ranks processed / the max-over-ranks time (weak scaling, no collective
    on the data path)."""
    return world * flops_per_rank_step / (ms_per_step * 1e-3) / 1e12


def replica_seed(base_seed: int, rank: int) -> int:
    """Each replica runs the same-shaped problem on its own seeded z."""
    return base_seed + rank


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
                pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        # median over the busier half of the samples (the sampler also sees idle gaps)
        load = sm[len(sm) // 2:] if sm else []
        med = load[len(load) // 2] if load else None
        return {"sm_mhz": med, "sm_max_mhz": mx, "power_w_max": max(pw) if pw else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# oracle legs (the ONLY places bench.py may execute oracle/): cpu_baseline and --impl reference
# ------------------------------------------------------------------------------------------------
def subgrid_flops(N: int, ni: int, nj: int) -> float:
    """Counted FLOPs of the sub-grid oracle on |I| x |J| output pairs (same counting rule as the
    full op: matmul FLOPs only)."""
    proj = 2.0 * (ni + nj) * N * C * (2 * C)          # a-pair on I rows, b-pair on J rows
    contr = 2.0 * C * ni * nj * N
    tail = 2.0 * ni * nj * C * C * 2                  # gate + output projection on I x J
    return proj + contr + tail


def oracle_sample_step(N: int, rows: int, seed: int, direction: int):
    """One bounded sample of the workload through the oracle as it stands: exact out[I x J] for
    `rows` x `rows` sampled pairs of the N-token problem (full sums over k)."""
    import numpy as np
    import torch
    from oracle import trimul_oracle as orc
    from paper_2603_14806_b200 import synth
    za, zb, zij = synth.make_z_slices(seed, rows, N, C, "bf16")
    p = synth.make_params(seed * 2 + direction, C, C, "bf16")
    f = lambda t: t.double().numpy()
    t0 = time.perf_counter()
    out = orc.trimul_subgrid(f(za), None, f(zb), None, f(zij), None, {k: f(v) for k, v in p.items()})
    dt = time.perf_counter() - t0
    assert np.all(np.isfinite(out))
    return dt


def host_info():
    """CPU model string, cores this process may run on, and the thread count numpy's BLAS really uses."""
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    blas_threads = None
    try:
        import numpy  # noqa: F401  (load the BLAS before asking)
        from threadpoolctl import threadpool_info
        blas = [d for d in threadpool_info() if d.get("user_api") == "blas"]
        if blas:
            blas_threads = max(int(d.get("num_threads", 0)) for d in blas)
    except Exception:
        pass
    return {"cpu_model": model, "cores_available": cores, "blas_threads": blas_threads or cores}


def oracle_full_op(N: int, direction: int, threads=None, split=False):
    """Wall-clock of the oracle's full op (orc.trimul as it stands) on the headline-shaped problem at N
    tokens (z ~ N(0,1) rounded to bf16, all-ones mask).  threads=1 pins the BLAS to one thread.
    split=True also times orc.contraction alone on the same a, b (for the labelled extrapolation)."""
    import contextlib
    import numpy as np
    from oracle import trimul_oracle as orc
    from paper_2603_14806_b200 import synth
    z = synth.make_z(7, N, C, "bf16", "cpu").double().numpy()
    p = {k: v.double().numpy() for k, v in synth.make_params(14 + direction, C, C, "bf16").items()}
    ctx = contextlib.nullcontext()
    if threads is not None:
        from threadpoolctl import threadpool_limits
        ctx = threadpool_limits(limits=threads)
    with ctx:
        t0 = time.perf_counter()
        out = orc.trimul(z, None, p, direction)
        dt = time.perf_counter() - t0
        assert np.all(np.isfinite(out))
        del out
        t_c = None
        if split:
            a, b = orc.projections(z, None, p)
            t0 = time.perf_counter()
            orc.contraction(a, b, direction)
            t_c = time.perf_counter() - t0
    return dt, t_c


def cpu_baseline_protocol(N_headline: int, budget_s: float):
    """SURVEY 8(d) "Oracle timed beside it": the oracle's FULL op wall-clocked at N = 64, 512 and 2048
    (N = 2048 once, and only if the N = 512 timing predicts it fits the budget and the host has the
    memory; otherwise N = 1024 and said so), one single-thread figure at N = 512, and the N = 4096
    figure as a LABELLED extrapolation (contraction ~ N^3, the rest ~ N^2)."""
    import psutil
    info = host_info()
    fl = lambda n: counted_flops(n)
    res = {"host": info, "full_op": {}}
    split512 = None
    for n in (64, 512):
        t_out, t_c = oracle_full_op(n, 0, split=(n == 512))
        t_in, _ = oracle_full_op(n, 1)
        if n == 512:
            split512 = (t_out, t_c)
        res["full_op"][f"N={n}"] = {"seconds_outgoing": t_out, "seconds_incoming": t_in,
                                     "tflops": 2 * fl(n) / (t_out + t_in) / 1e12,
                                     "threads": info["blas_threads"]}
    t1, _ = oracle_full_op(512, 0, threads=1)
    res["single_thread"] = {"N": 512, "direction": "outgoing", "seconds": t1, "tflops": fl(512) / t1 / 1e12}
    # largest of N = 2048 / 1024 whose predicted time (contraction ~ N^3, the rest ~ N^2, from the
    # N = 512 split) fits the budget and whose fp64 working set (~12 arrays of N*N*128 doubles) fits
    predict = lambda n: split512[1] * (n / 512) ** 3 + (split512[0] - split512[1]) * (n / 512) ** 2
    big = 1024
    if predict(2048) <= budget_s and psutil.virtual_memory().available > 12 * 2048 * 2048 * C * 8 * 1.2:
        big = 2048
    t_big, t_contr = oracle_full_op(big, 0, split=True)
    res["full_op"][f"N={big}"] = {"seconds_outgoing": t_big, "seconds_contraction_alone": t_contr,
                                   "tflops": fl(big) / t_big / 1e12, "threads": info["blas_threads"],
                                   "note": "timed once (outgoing)" + ("" if big == 2048 else
                                           f"; N=2048 was predicted at {predict(2048):.0f} s, over the "
                                           f"{budget_s:.0f} s budget of the default run (--cpu-budget)")}
    r = N_headline / big
    t_head = t_contr * r ** 3 + (t_big - t_contr) * r ** 2
    res["extrapolated"] = {"N": N_headline, "seconds_per_call": t_head, "tflops": fl(N_headline) / t_head / 1e12,
                           "label": f"EXTRAPOLATION from the measured N={big} full op: contraction x{r:g}^3, "
                                    f"the rest x{r:g}^2 -- not measured"}
    res["value"] = res["full_op"][f"N={big}"]["tflops"]
    res["unit"] = "TFLOP/s"
    res["cores"] = info["blas_threads"]
    res["kind"] = "oracle"
    res["sample"] = (f"fp64 numpy oracle, FULL op at N={big} (outgoing, timed once) on {info['blas_threads']} BLAS "
                     f"threads of {info['cpu_model']}; full-op timings at N=64 / 512 (both directions), a "
                     f"single-thread figure at N=512 and a labelled extrapolation to N={N_headline} beside it")
    return res


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    N, rows = args.n, args.ref_rows
    # the oracle has no caches or lazy initialisation worth more than one untimed call: ONE warm-up
    # sample whatever --warmup says (stated in the line as warmup_run)
    warm = min(args.warmup, 1)
    for _ in range(warm):
        oracle_sample_step(N, rows, 0, 0)
    times = []
    for s in range(args.steps):
        times.append(oracle_sample_step(N, rows, 10 + s, 0) + oracle_sample_step(N, rows, 10 + s, 1))
    total = sum(times)
    fl = 2 * subgrid_flops(N, rows, rows) * args.steps
    val = fl / total / 1e12
    info = host_info()
    cores = info["blas_threads"]
    sample = (f"sub-grid oracle, {rows}x{rows} sampled output pairs of the N={N} problem (exact full-k "
              f"sums), outgoing+incoming per step; TFLOP/s on the sample's own counted FLOPs")
    line = {
        "impl": "reference", "metric": "triangle-mult TFLOP/s at N=4096 c=128 bf16 (outgoing+incoming)",
        "value": val, "unit": "TFLOP/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "warmup_run": warm, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "host": info,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE configs[3]: trimul outgoing+incoming N={N} c_z=c=128 all-ones mask",
                   "sample": sample},
        "cpu_baseline": {"value": val, "unit": "TFLOP/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2603_14806_b200 import binding as B
    from paper_2603_14806_b200 import build as builder
    from paper_2603_14806_b200 import synth

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        builder.build()
    if world > 1:
        dist.barrier()
    B.load()

    N, K, W = args.n, args.steps, max(args.warmup, 3)
    cfg = synth.CONFIGS[3]
    # replicas: every rank runs the same-shaped problem on its own seeded inputs
    z = synth.make_z(replica_seed(cfg.seed, rank), N, C, "bf16", dev)
    M = synth.pair_mask(synth.make_token_mask("ones", N, cfg.seed), "bf16", dev)
    ps = [{k: v.to(dev) for k, v in synth.make_params(cfg.seed * 2 + d, C, C, "bf16").items()}
          for d in (0, 1)]
    ws = torch.empty(B.workspace_bytes(N), dtype=torch.uint8, device=dev)
    outs = [torch.empty_like(z), torch.empty_like(z)]

    def step():
        B.trimul(z, M, ps[0], B.OUTGOING, out=outs[0], workspace=ws)
        B.trimul(z, M, ps[1], B.INCOMING, out=outs[1], workspace=ws)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(W):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(K):
        step()
    e1.record()
    barrier()
    ms = max_over_ranks(e0.elapsed_time(e1), world, dist, dev)
    ms_per_step = ms / K
    flops_step = 2 * counted_flops(N)
    value = whole_job_tflops(flops_step, ms_per_step, world)

    # ---- per-stage durations inside a timed region: the stages in the form foldcp_trimul chains them
    # (project_stats -> contract with fp16 scaled o -> finalize_fused: bitwise the fused call, see
    # tests/test_parity_gpu.py test_fused_stage_chain_is_the_full_call_bitwise), same stream
    tb = C * N * N * 2
    a = ws[:tb].view(torch.float16).view(C, N, N)
    b = ws[tb: 2 * tb].view(torch.float16).view(C, N, N)
    o = ws[2 * tb: 3 * tb].view(torch.float16).view(C, N, N)
    zst = ws[3 * tb: 3 * tb + N * N * 8].view(torch.float32).view(N, N, 2)
    scratch = B.stage_scratch(dev)
    import ctypes
    lib = B.load()
    stream = torch.cuda.current_stream().cuda_stream
    stage_ms = {"k1": 0.0, "k2_out": 0.0, "k2_in": 0.0, "k3": 0.0}
    evs = []
    for it in range(K):
        for d in (0, 1):
            prm = B.make_params(ps[d], B.BF16, 1e-5, True)
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            ev[0].record()
            st = lib.foldcp_trimul_project_stats(z.data_ptr(), M.data_ptr(), ctypes.byref(prm), N, C, C,
                                                 a.data_ptr(), b.data_ptr(), zst.data_ptr(),
                                                 scratch.data_ptr(), stream)
            ev[1].record()
            st |= lib.foldcp_trimul_contract(a.data_ptr(), b.data_ptr(), N, C, B.BF16_F16ALL, d,
                                             o.data_ptr(), scratch.data_ptr(), stream)
            ev[2].record()
            st |= lib.foldcp_trimul_finalize_fused(o.data_ptr(), z.data_ptr(), zst.data_ptr(), M.data_ptr(),
                                                   ctypes.byref(prm), N, C, C, outs[d].data_ptr(), stream)
            ev[3].record()
            assert st == 0
            evs.append((d, ev))
    torch.cuda.synchronize()
    for d, ev in evs:
        stage_ms["k1"] += ev[0].elapsed_time(ev[1])
        stage_ms["k2_out" if d == 0 else "k2_in"] += ev[1].elapsed_time(ev[2])
        stage_ms["k3"] += ev[2].elapsed_time(ev[3])
    # ---- per-direction ms: events around each foldcp_trimul call, same loop length
    dir_ev = []
    for it in range(K):
        for d in (0, 1):
            e_a, e_b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e_a.record()
            B.trimul(z, M, ps[d], d, out=outs[d], workspace=ws)
            e_b.record()
            dir_ev.append((d, e_a, e_b))
    torch.cuda.synchronize()
    per_direction = {"outgoing": sum(a.elapsed_time(b) for d, a, b in dir_ev if d == 0) / K,
                     "incoming": sum(a.elapsed_time(b) for d, a, b in dir_ev if d == 1) / K}
    clocks = sampler.stop() if rank == 0 else None
    stage_ms["k1"] /= 2 * K
    stage_ms["k3"] /= 2 * K
    stage_ms["k2_out"] /= K
    stage_ms["k2_in"] /= K
    return dict(torch=torch, dist=dist, B=B, synth=synth, rank=rank, world=world, dev=dev, N=N, K=K,
                W=W, z=z, M=M, ps=ps, ws=ws, outs=outs, ms_per_step=ms_per_step, value=value,
                stage_ms=stage_ms, clocks=clocks, flops_step=flops_step, per_direction=per_direction)


def run_backward(ctx, steps):
    """NEXT-2: the full backward pass (foldcp_trimul_backward) at the headline size, both directions,
    CUDA events around each call.  FLOPs counted: the forward recomputation (one forward call), the
    two contraction-gradient GEMMs (2 x 2cN^3) and the 12 projection-sized GEMMs of the tail
    (6 data gradients + 6 weight gradients, 2 N^2 c^2 each)."""
    torch, B = ctx["torch"], ctx["B"]
    z, M, ps, dev, N = ctx["z"], ctx["M"], ctx["ps"], ctx["dev"], ctx["N"]
    ws = torch.empty(B.backward_workspace_bytes(N), dtype=torch.uint8, device=dev)
    g = torch.Generator(device=dev).manual_seed(77)
    d_out = torch.empty_like(z)
    for r0 in range(0, N, 256):
        d_out[r0:r0 + 256] = torch.randn(min(256, N - r0), N, C, generator=g, device=dev).to(z.dtype)
    res = {}
    for d, name in ((0, "outgoing"), (1, "incoming")):
        B.trimul_backward(d_out, z, M, ps[d], d, workspace=ws)          # warm-up
        torch.cuda.synchronize()
        evs = []
        for _ in range(steps):
            e_a, e_b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e_a.record()
            B.trimul_backward(d_out, z, M, ps[d], d, workspace=ws)
            e_b.record()
            evs.append((e_a, e_b))
        torch.cuda.synchronize()
        res[name] = sum(a.elapsed_time(b) for a, b in evs) / steps
    fl = counted_flops(N) + 2 * 2.0 * C * N ** 3 + 12 * 2.0 * N * N * C * C
    ms = 0.5 * (res["outgoing"] + res["incoming"])
    del ws, d_out
    torch.cuda.empty_cache()
    return {"ms_per_call": res, "counted_tflop_per_call": fl / 1e12, "tflops": fl / (ms * 1e-3) / 1e12,
            "steps": steps, "workspace_bytes": B.backward_workspace_bytes(N),
            "note": "forward recomputation + contraction gradients on tcgen05; LayerNorm / gate / projection "
                    "backward and weight gradients on fp32 CUDA-core kernels (first correct path)"}


def run_triattn(ctx, N=1024, steps=2):
    """NEXT-4: triangle attention (foldcp_triattn), starting and ending node, bf16 storage, on a
    synthetic pair tensor of N tokens (mask: last 10 % of tokens padding).  Counted FLOPs: QK^T and PV
    (4 N^3 H c) plus the projections (oracle/triattn_oracle.py flops())."""
    torch, B, synth = ctx["torch"], ctx["B"], ctx["synth"]
    dev = ctx["dev"]
    g = torch.Generator(device=dev).manual_seed(4242)
    rn = lambda *s: torch.randn(*s, generator=g, device=dev)
    z = rn(N, N, C).to(torch.bfloat16)
    p = dict(ln_gamma=1 + 0.1 * rn(C), ln_beta=0.1 * rn(C))
    for name, rows in (("w_q", C), ("w_k", C), ("w_v", C), ("w_g", C), ("w_t", 4)):
        p[name] = (rn(rows, C) / C ** 0.5).to(torch.bfloat16)
    p["w_o"] = (rn(C, C) / C ** 0.5).to(torch.bfloat16)
    m = synth.make_token_mask("tail", N, 7)
    M = synth.pair_mask(m, "bf16", dev)
    M[:, 0] = 1
    M[0, :] = 1
    ws = torch.empty(B.triattn_workspace_bytes(N), dtype=torch.uint8, device=dev)
    out = torch.empty_like(z)
    res = {}
    for node, name in ((B.TRIATTN_STARTING, "starting"), (B.TRIATTN_ENDING, "ending")):
        B.triattn(z, M, p, node, out=out, workspace=ws)
        torch.cuda.synchronize()
        e_a, e_b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e_a.record()
        for _ in range(steps):
            B.triattn(z, M, p, node, out=out, workspace=ws)
        e_b.record()
        torch.cuda.synchronize()
        res[name] = e_a.elapsed_time(e_b) / steps
    fl = 4.0 * N ** 3 * C + 2.0 * N * N * C * (4 * C + 4) + 2.0 * N * N * C * C
    ms = 0.5 * (res["starting"] + res["ending"])
    del z, M, ws, out
    torch.cuda.empty_cache()
    return {"workload": f"triangle attention (PAPER.md Eq. 1), N={N}, c_z=128, 4 heads x 32, bf16 storage",
            "ms_per_call": res, "counted_tflop_per_call": fl / 1e12, "tflops": fl / (ms * 1e-3) / 1e12,
            "steps": steps, "gpu_launches_per_call": 3,
            "note": "bf16 mode: projections, QK^T, PV and the output projection on tcgen05 (csrc/triattn.cu)"}


def run_n8192(ctx, steps=3):
    """BASELINE configs[4] (N = 8192, 5 % of tokens masked) in a single call per direction: 3 timed
    calls each, CUDA events; peak HBM bytes from torch's allocator."""
    torch, B, synth = ctx["torch"], ctx["B"], ctx["synth"]
    dev, ps = ctx["dev"], ctx["ps"]
    free, _ = torch.cuda.mem_get_info()
    N = 8192
    need = 2 * N * N * C * 2 + B.workspace_bytes(N)
    if free < need + (4 << 30):
        return {"skipped": f"needs {need / 2**30:.0f} GiB of free HBM, {free / 2**30:.0f} GiB free"}
    cfg = synth.CONFIGS[4]
    torch.cuda.reset_peak_memory_stats(dev)
    base = torch.cuda.memory_allocated(dev)
    z = synth.make_z(cfg.seed, N, C, "bf16", dev)
    M = synth.pair_mask(synth.make_token_mask(cfg.mask_kind, N, cfg.seed), "bf16", dev)
    ws = torch.empty(B.workspace_bytes(N), dtype=torch.uint8, device=dev)
    out = torch.empty_like(z)
    res = {}
    for d, name in ((0, "outgoing"), (1, "incoming")):
        B.trimul(z, M, ps[d], d, out=out, workspace=ws)                   # warm-up
        torch.cuda.synchronize()
        evs = []
        for _ in range(steps):
            e_a, e_b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e_a.record()
            B.trimul(z, M, ps[d], d, out=out, workspace=ws)
            e_b.record()
            evs.append((e_a, e_b))
        torch.cuda.synchronize()
        res[name] = sum(a.elapsed_time(b) for a, b in evs) / steps
    peak = torch.cuda.max_memory_allocated(dev) - base
    ms = 0.5 * (res["outgoing"] + res["incoming"])
    del z, M, ws, out
    torch.cuda.empty_cache()
    return {"workload": "BASELINE configs[4]: N=8192, 5 % of tokens masked, single call per direction",
            "ms_per_call": res, "tflops": counted_flops(N) / (ms * 1e-3) / 1e12,
            "counted_tflop_per_call": counted_flops(N) / 1e12, "steps": steps,
            "peak_hbm_bytes": int(peak), "peak_hbm_GiB": peak / 2 ** 30}


def run_e2e(ctx, steps):
    """Same metric end to end: every step copies z and the mask from pinned host memory, runs both
    directions through the public binding and reads both results back to pinned host memory.
    The three legs run on their own streams with double-buffered device tensors, so step i+1's
    upload and step i-1's download overlap step i's kernels (PCIe is full duplex); every step
    still moves its own 4.3 GB in and 8.6 GB out inside the timed region."""
    torch, B = ctx["torch"], ctx["B"]
    z, M, ps, ws, dev = ctx["z"], ctx["M"], ctx["ps"], ctx["ws"], ctx["dev"]
    hz = torch.empty(z.shape, dtype=z.dtype, pin_memory=True)
    hM = torch.empty(M.shape, dtype=M.dtype, pin_memory=True)
    hz.copy_(z)
    hM.copy_(M)
    ho = [torch.empty(z.shape, dtype=z.dtype, pin_memory=True) for _ in range(2)]
    dz = [torch.empty_like(z) for _ in range(2)]
    dM = [torch.empty_like(M) for _ in range(2)]
    douts = [[torch.empty_like(z), torch.empty_like(z)] for _ in range(2)]
    s_in, s_cmp, s_out = (torch.cuda.Stream(device=dev) for _ in range(3))
    ev_in = [torch.cuda.Event() for _ in range(2)]
    ev_cmp = [torch.cuda.Event() for _ in range(2)]
    ev_out = [torch.cuda.Event() for _ in range(2)]

    def step(i):
        b = i & 1
        with torch.cuda.stream(s_in):
            s_in.wait_event(ev_cmp[b])            # dz[b] was read by step i-2's kernels
            dz[b].copy_(hz, non_blocking=True)
            dM[b].copy_(hM, non_blocking=True)
            ev_in[b].record(s_in)
        with torch.cuda.stream(s_cmp):
            s_cmp.wait_event(ev_in[b])
            s_cmp.wait_event(ev_out[b])           # douts[b] was downloaded by step i-2
            B.trimul(dz[b], dM[b], ps[0], B.OUTGOING, out=douts[b][0], workspace=ws)
            B.trimul(dz[b], dM[b], ps[1], B.INCOMING, out=douts[b][1], workspace=ws)
            ev_cmp[b].record(s_cmp)
        with torch.cuda.stream(s_out):
            s_out.wait_event(ev_cmp[b])
            ho[0].copy_(douts[b][0], non_blocking=True)
            ho[1].copy_(douts[b][1], non_blocking=True)
            ev_out[b].record(s_out)

    torch.cuda.synchronize()
    for i in range(2):
        step(i)                                   # warm-up, also arms every event once
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(s_in)
    for i in range(steps):
        step(i)
    s_out.wait_stream(s_cmp)
    s_out.wait_stream(s_in)
    e1.record(s_out)
    torch.cuda.synchronize()
    ms = max_over_ranks(e0.elapsed_time(e1) / steps, ctx["world"], ctx["dist"], dev)
    h2d = hz.numel() * hz.element_size() + hM.numel() * hM.element_size()
    d2h = 2 * ho[0].numel() * ho[0].element_size()
    return {"value": whole_job_tflops(ctx["flops_step"], ms, ctx["world"]), "unit": "TFLOP/s",
            "ms_per_step": ms, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": steps,
            "overlap": "upload / kernels / download on three streams, double-buffered"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=4096, help="tokens (default: BASELINE configs[3])")
    ap.add_argument("--ref-rows", type=int, default=128,
                    help="sub-grid size of the oracle sample (128: ~12 s of CPU work per step)")
    ap.add_argument("--cpu-budget", type=float, default=90.0,
                    help="seconds the N=2048 full-op oracle timing may take (else N=1024 is timed)")
    ap.add_argument("--no-n8192", action="store_true")
    ap.add_argument("--no-backward", action="store_true")
    ap.add_argument("--no-triattn", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return

    ctx = run_ours(args)
    N, K, world = ctx["N"], ctx["K"], ctx["world"]
    e2e = None if args.no_e2e else run_e2e(ctx, max(4, min(K, 6)))
    single = world == 1 and ctx["rank"] == 0
    bwd = run_backward(ctx, 2) if (single and not args.no_backward) else None
    triattn = run_triattn(ctx) if (single and not args.no_triattn) else None
    n8192 = None
    if single and not args.no_n8192:
        for k in ("z", "M", "ws", "outs"):
            ctx[k] = None
        ctx["torch"].cuda.empty_cache()
        n8192 = run_n8192(ctx)
    if ctx["rank"] != 0:
        if world > 1:
            ctx["dist"].barrier()
            ctx["dist"].destroy_process_group()
        return
    peaks = measured_peaks()
    sm = ctx["stage_ms"]
    k2_ms = 0.5 * (sm["k2_out"] + sm["k2_in"])
    k2_tf = 2.0 * C * N ** 3 / (k2_ms * 1e-3) / 1e12
    step_sum = 2 * sm["k1"] + sm["k2_out"] + sm["k2_in"] + 2 * sm["k3"]
    traffic, traffic_file = k2_traffic_from_profile()
    roofline = {
        "bound": "tensor", "kernel": "k2_contract_kernel (mean of outgoing and incoming launches)",
        "achieved": k2_tf, "peak": peaks["tf_sustained"], "unit": "TFLOP/s",
        "frac": k2_tf / peaks["tf_sustained"],
        "peak_kind": f"{peaks['source']} cuBLAS bf16, sustained figure (kernel timed inside a long step)",
        "frac_of_burst_peak": k2_tf / peaks["tf_burst"], "peak_burst": peaks["tf_burst"],
        "frac_of_datasheet_2250": k2_tf / 2250.0,
        "algorithmic_flops_per_launch": 2.0 * C * N ** 3,
        "ms_per_launch": {"outgoing": sm["k2_out"], "incoming": sm["k2_in"]},
        "share_of_step": (sm["k2_out"] + sm["k2_in"]) / step_sum,
        # dram__bytes_read.sum + dram__bytes_write.sum of one k2_contract launch at N=4096, parsed
        # from the newest ncu --set full summary under profiles/ (null if there is none)
        "traffic": traffic if N == 4096 else None,
        "traffic_source": None if traffic_file is None else "profiles/" + traffic_file,
        "algorithmic_bytes_per_launch": 3.0 * C * N * N * 2,
        "other_kernels": {
            "k1_project": {"ms": sm["k1"], "bound": "hbm",
                           "achieved_GBs": 3 * N * N * C * 2 / (sm["k1"] * 1e-3) / 1e9,
                           "frac": 3 * N * N * C * 2 / (sm["k1"] * 1e-3) / 1e9 / peaks["hbm_gbs"]},
            "k3_finalize": {"ms": sm["k3"], "bound": "hbm",
                            "achieved_GBs": 3 * N * N * C * 2 / (sm["k3"] * 1e-3) / 1e9,
                            "frac": 3 * N * N * C * 2 / (sm["k3"] * 1e-3) / 1e9 / peaks["hbm_gbs"]},
        },
    }
    cpu = None
    if not args.no_cpu_baseline:
        cpu = cpu_baseline_protocol(N, args.cpu_budget)
    line = {
        "metric": "triangle-mult TFLOP/s at N=4096 c=128 bf16 (outgoing+incoming)",
        "value": ctx["value"], "unit": "TFLOP/s", "n_gpus": world, "steps": K, "warmup": ctx["W"],
        "ms_per_step": ctx["ms_per_step"], "ms_per_call": ctx["ms_per_step"] / 2,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": {"workload": f"BASELINE configs[3]: trimul outgoing+incoming, N={N}, c_z=c_hidden=128, "
                               "bf16 in / fp32 accumulate, all-ones pair mask, batch 1",
                   "l2": "inputs (4 GiB z, 12 GiB workspace) exceed the 126 MB L2; no flush needed",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "counted_tflop_per_step": ctx["flops_step"] / 1e12},
        "frac_of_peak": {"measured_burst": ctx["value"] / world / peaks["tf_burst"],
                         "measured_sustained": ctx["value"] / world / peaks["tf_sustained"],
                         "datasheet_2250": ctx["value"] / world / 2250.0},
        "clocks": ctx["clocks"], "e2e": e2e, "gpu_launches": 3 * 2 * K,
        "roofline": roofline, "cpu_baseline": cpu,
        "per_direction": {"ms_per_call": ctx["per_direction"],
                          "tflops": {k: counted_flops(N) / (v * 1e-3) / 1e12
                                     for k, v in ctx["per_direction"].items()}},
        "n8192": n8192, "backward": bwd, "triattn": triattn,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        ctx["dist"].barrier()
        ctx["dist"].destroy_process_group()


if __name__ == "__main__":
    main()
