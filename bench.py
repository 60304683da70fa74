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
K2_DRAM_BYTES_PER_LAUNCH_N4096 = 9.06e9 + 4.28e9   # ncu, profiles/r1_k2_contract_ncu_full.txt


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


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    N, rows = args.n, args.ref_rows
    for _ in range(min(args.warmup, 1)):
        oracle_sample_step(N, rows, 0, 0)
    times = []
    for s in range(args.steps):
        times.append(oracle_sample_step(N, rows, 10 + s, 0) + oracle_sample_step(N, rows, 10 + s, 1))
    total = sum(times)
    fl = 2 * subgrid_flops(N, rows, rows) * args.steps
    val = fl / total / 1e12
    cores = os.cpu_count()
    sample = (f"sub-grid oracle, {rows}x{rows} sampled output pairs of the N={N} problem (exact full-k "
              f"sums), outgoing+incoming per step; TFLOP/s on the sample's own counted FLOPs")
    line = {
        "impl": "reference", "metric": "triangle-mult TFLOP/s at N=4096 c=128 bf16 (outgoing+incoming)",
        "value": val, "unit": "TFLOP/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True,
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

    # ---- per-stage durations inside a timed region (stage entry points, same kernels, same stream)
    tb = C * N * N * 2
    a = ws[:tb].view(torch.bfloat16).view(C, N, N)
    b = ws[tb: 2 * tb].view(torch.bfloat16).view(C, N, N)
    o = ws[2 * tb: 3 * tb].view(torch.bfloat16).view(C, N, N)
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
            st = lib.foldcp_trimul_project(z.data_ptr(), M.data_ptr(), ctypes.byref(prm), N, C, C,
                                           a.data_ptr(), b.data_ptr(), scratch.data_ptr(), stream)
            ev[1].record()
            st |= lib.foldcp_trimul_contract(a.data_ptr(), b.data_ptr(), N, C, B.BF16, d,
                                             o.data_ptr(), scratch.data_ptr(), stream)
            ev[2].record()
            st |= lib.foldcp_trimul_finalize(o.data_ptr(), z.data_ptr(), M.data_ptr(),
                                             ctypes.byref(prm), N, C, C, outs[d].data_ptr(), stream)
            ev[3].record()
            assert st == 0
            evs.append((d, ev))
    torch.cuda.synchronize()
    for d, ev in evs:
        stage_ms["k1"] += ev[0].elapsed_time(ev[1])
        stage_ms["k2_out" if d == 0 else "k2_in"] += ev[1].elapsed_time(ev[2])
        stage_ms["k3"] += ev[2].elapsed_time(ev[3])
    clocks = sampler.stop() if rank == 0 else None
    stage_ms["k1"] /= 2 * K
    stage_ms["k3"] /= 2 * K
    stage_ms["k2_out"] /= K
    stage_ms["k2_in"] /= K
    return dict(torch=torch, dist=dist, B=B, synth=synth, rank=rank, world=world, dev=dev, N=N, K=K,
                W=W, z=z, M=M, ps=ps, ws=ws, outs=outs, ms_per_step=ms_per_step, value=value,
                stage_ms=stage_ms, clocks=clocks, flops_step=flops_step)


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
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return

    ctx = run_ours(args)
    N, K, world = ctx["N"], ctx["K"], ctx["world"]
    e2e = None if args.no_e2e else run_e2e(ctx, max(4, min(K, 6)))
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
        # dram__bytes_read.sum + dram__bytes_write.sum of one k2_contract launch at N=4096, from the
        # ncu --set full capture summarised in profiles/ (9.06 GB read + 4.28 GB written; the
        # algorithmic bytes are 8.59 GB read + 4.29 GB written)
        "traffic": K2_DRAM_BYTES_PER_LAUNCH_N4096 if N == 4096 else None,
        "traffic_source": "profiles/r1_k2_contract_ncu_full.txt",
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
        rows = args.ref_rows
        t = oracle_sample_step(N, rows, 1, 0) + oracle_sample_step(N, rows, 1, 1)
        cpu = {"value": 2 * subgrid_flops(N, rows, rows) / t / 1e12, "unit": "TFLOP/s",
               "cores": os.cpu_count(), "kind": "oracle", "seconds": t,
               "sample": f"sub-grid oracle, {rows}x{rows} sampled output pairs of the N={N} problem, "
                         f"outgoing+incoming (exact full-k sums), fp64 numpy"}
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
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        ctx["dist"].barrier()
        ctx["dist"].destroy_process_group()


if __name__ == "__main__":
    main()
