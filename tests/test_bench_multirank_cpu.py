"""The N > 1 path of bench.py is "replicas only": no collective on the data
path, max-over-ranks timing, value = all ranks' FLOPs / that time.  world_size-2 gloo, CPU only."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    local_ms = 10.0 + 5.0 * rank            # rank 1 is the slow replica
    ms = bench.max_over_ranks(local_ms, world, dist, "cpu")
    flops = 2 * bench.counted_flops(4096)
    q.put((rank, ms, bench.whole_job_tflops(flops, ms, world), bench.replica_seed(1003, rank)))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_max_over_ranks_and_whole_job_value():
    import bench
    world, port = 2, 29500 + (os.getpid() % 1000)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    flops = 2 * bench.counted_flops(4096)
    for rank, ms, value, seed in res:
        assert ms == 15.0                                     # the slowest replica's time, on every rank
        assert abs(value - 2 * flops / 15e-3 / 1e12) < 1e-9   # both replicas' FLOPs over that time
        assert seed == 1003 + rank                            # per-replica inputs
    assert bench.max_over_ranks(7.0, 1) == 7.0                # single GPU: no process group needed


def test_counted_flops_is_baseline_md_figure():
    import bench
    assert abs(bench.counted_flops(4096) / 1e12 - 20.891) < 1e-3
