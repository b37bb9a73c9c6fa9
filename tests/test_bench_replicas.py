"""Multi-GPU host logic of bench.py on CPU: the path does not shard ("replicas only"), so N > 1 means N
independent replicas whose timings are reduced with MAX over ranks.  Two gloo processes exercise exactly the
functions bench.py uses for that (no GPU, no CUDA library needed)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        local_ms = 10.0 + 5.0 * rank                       # rank 1 is the slow replica
        ms = bench.max_over_ranks(local_ms, dist, torch.device("cpu"))
        value = bench.whole_job_value(world, 1000, 4, ms * 1e-3)
        # every rank must agree on the job-wide numbers
        t = torch.tensor([ms, value], dtype=torch.float64)
        gathered = [torch.zeros_like(t) for _ in range(world)]
        dist.all_gather(gathered, t)
        if rank == 0:
            out.put([g.tolist() for g in gathered])
    finally:
        dist.destroy_process_group()


def test_replica_timing_is_max_over_ranks_and_value_is_whole_job():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for ms, value in res:
        assert ms == 15.0                                  # the slow rank's time
        assert abs(value - 2 * 1000 * 4 / 15e-3) < 1e-6   # cells of BOTH replicas / max time


def test_single_process_path_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.whole_job_value(1, 10, 2, 0.5) == 40.0
    r = bench.fp64_roofline("config5_512", 512 ** 3, 9.0)
    assert r["bound"] == "alu" and 0.0 < r["frac"] < 1.0
    assert abs(r["peak"] - 64 * 148 * 1.965e9 / 1e12) < 1e-9
