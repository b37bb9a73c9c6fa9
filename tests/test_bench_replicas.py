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
    c = {"kernel_rev": "rX", "fp64_instr_per_cell": 400.0, "dram_bytes_per_launch": 1.1e10, "source": "profiles/x.md"}
    r = bench.fp64_roofline(c, 512 ** 3, 9.0)
    assert r["bound"] == "alu" and 0.0 < r["frac"] < 1.0
    assert abs(r["peak"] - 64 * 148 * 1.965e9 / 1e12) < 1e-9           # nominal peak when none was measured
    r = bench.fp64_roofline(c, 512 ** 3, 9.0, 17.0, "measured")
    assert r["peak"] == 17.0 and r["peak_source"] == "measured"
    assert bench.fp64_roofline(None, 512 ** 3, 9.0) is None


def test_ncu_counters_in_profiles_belong_to_the_built_kernels():
    """bench.py prints roofline.traffic and fp64 instructions per cell from profiles/r03_step_kernel_counters.csv; the
    rows must have been captured for the kernel revision the library reports (ark_version_string needs no GPU), and a
    row of another revision must be ignored instead of being printed as if it were current."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_1903_09043_b200 import binding
    version = binding.version_string()
    rev = bench.kernel_rev(version)
    assert rev, version
    table = bench.load_counters()
    cells = {"config5_512": (512 ** 3, 80.0), "config4_256": (256 ** 3, 80.0), "inviscid3d_512": (512 ** 3, 80.0),
             "config4_256_phi": (256 ** 3, 88.0)}
    for name in sorted(cells):
        assert name in table, "no ncu counters committed for %s" % name
        assert table[name]["kernel_rev"] == rev, (name, table[name]["kernel_rev"], rev)
        assert os.path.exists(os.path.join(ROOT, table[name]["source"]))
        c = bench.counters_for(name, version, table)
        assert c is not None and 200.0 < c["fp64_instr_per_cell"] < 600.0
        ncell, bpc = cells[name]
        assert 1.0 <= c["dram_bytes_per_launch"] / (bpc * ncell) < 1.3           # DRAM traffic close to the algorithmic bytes per cell
    stale = {"config5_512": dict(table["config5_512"], kernel_rev="r0.0")}
    assert bench.counters_for("config5_512", version, stale) is None


def test_gpus_flag_spawns_its_own_ranks(monkeypatch):
    """`python bench.py --gpus N` outside torchrun re-launches itself under torch.distributed.run with N ranks on
    127.0.0.1 (so n_gpus in the JSON line is what actually ran)."""
    sys.path.insert(0, ROOT)
    import argparse
    import bench
    seen = {}
    monkeypatch.setattr(bench.subprocess, "call", lambda cmd: seen.setdefault("cmd", cmd) and 0)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "4", "--steps", "2"])
    assert bench.spawn_ranks(argparse.Namespace(gpus=4)) == 0
    cmd = seen["cmd"]
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node" in cmd and cmd[cmd.index("--nproc-per-node") + 1] == "4"
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[-4:] == ["--gpus", "4", "--steps", "2"]


def test_two_ranks_launched_by_torch_distributed_run(tmp_path):
    """The launch line bench.py builds (torch.distributed.run, 2 ranks, 127.0.0.1) with a gloo worker that uses bench's
    own reductions: both ranks must report the slow rank's time."""
    import subprocess
    worker = tmp_path / "worker.py"
    worker.write_text(
        "import os, sys, torch, torch.distributed as dist\n"
        "sys.path.insert(0, %r)\n"
        "import bench\n"
        "dist.init_process_group('gloo')\n"
        "r = dist.get_rank()\n"
        "ms = bench.max_over_ranks(10.0 + 5.0 * r, dist, torch.device('cpu'))\n"
        "open(os.path.join(%r, 'rank%%d.txt' %% r), 'w').write('%%r %%r' %% (ms, bench.whole_job_value(dist.get_world_size(), 1000, 4, ms * 1e-3)))\n"
        "dist.destroy_process_group()\n" % (ROOT, str(tmp_path)))
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
                          "127.0.0.1", "--master-port", str(_free_port()), str(worker)], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [(str(r),) + tuple((tmp_path / ("rank%d.txt" % r)).read_text().split()) for r in range(2)]   # (one file per rank: their stdout interleaves)
    for ln in lines:
        assert float(ln[1]) == 15.0 and abs(float(ln[2]) - 2 * 1000 * 4 / 15e-3) < 1e-6
