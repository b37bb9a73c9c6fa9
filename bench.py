#!/usr/bin/env python
"""bench.py -- cell-updates/s of the full ARK time step (compute_dt + step) on B200, with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one pass of the whole hot path over the synthetic workload: ghost fill (y, z sweeps; the periodic x ghost
columns are written by the step kernel itself), fused acoustic+transport+dissipative+update kernel with the CFL
epilogue, the second reduction pass and the 16-byte device->host read of dt (ark_compute_dt) -- exactly the loop
{dt = ark_compute_dt(cfl); ark_step(dt)}.

The JSON line of the default workload (config5_512) also carries, under "also" (a list), the same measurement of the other
roofline target of north_star (config4_256), of the kernel variants no BASELINE config selects (inviscid3d_512: <VISC=0>;
config4_256_phi: the general path with an array-valued potential, 88 B per cell update) and of the three 2D BASELINE
configs (host loop and ark_run), each with its own clocks record.  The fp64 peak of the "alu" roofline is MEASURED in the same run
(ark_measure_fp64_peak: DFMA chains); the ncu-derived per-cell counters come from profiles/r03_step_kernel_counters.csv
and are only reported when that file was captured for the kernel revision of the loaded library.

Multi-GPU: the path does not shard in this build ("replicas only"): --gpus N runs N independent
replicas of the workload, one process per GPU, no data-path collective; value = N * cells * K / max time.  Started
without a torchrun environment, `--gpus N` (N > 1) re-launches itself under torch.distributed.run with N ranks.
"""
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

METRIC = "cell-updates/sec per full time step (fp64)"
UNIT = "cell-updates/s"
CFL = 0.4

WORKLOADS = {
    # name: (builder name in inputs, n, bytes per cell update, oracle sample size)
    "config5_512": ("config5_convection3d", 512, 80, 256),     # oracle sample: 256^3 (~6 s per step on one core)
    "config4_256": ("config4_rb3d", 256, 80, 256),
    "config3_1024x512": ("config3_rb2d", (1024, 512), 64, (512, 256)),
    "config2_512": ("config2_gresho", 512, 64, 512),
    "config1_128": ("config1_atmosphere", 128, 64, 128),
    # kernel variants that no BASELINE config selects (they ride along under "also"): the Euler part
    # alone (<VISC=0>) and the general path with an array-valued potential (<GEN=1>, 88 B per cell update)
    "inviscid3d_512": ("inviscid_convection3d", 512, 80, 256),
    "config4_256_phi": ("config4_rb3d_phi", 256, 88, 128),
}
# measured in the same line as the default workload: (name, timed steps of the host loop, ark_run steps or 0)
ALSO = [("config4_256", 20, 0), ("inviscid3d_512", 10, 0), ("config4_256_phi", 20, 0),
        ("config3_1024x512", 200, 2000), ("config2_512", 200, 2000), ("config1_128", 200, 2000)]


def build_workload(name, device=None, sample=False):
    from paper_1903_09043_b200 import inputs
    fn, n, bpc, ns = WORKLOADS[name]
    size = ns if sample else n
    f = getattr(inputs, fn)
    if isinstance(size, tuple):
        prm, U = f(size[0], size[1], device=device)
    else:
        prm, U = f(size, device=device)
    return prm, U, bpc


# fp64 ALU roof: measured in the same run by a register-resident DFMA-chain kernel of the library
# (ark_measure_fp64_peak).  For context: 64 fp64 instructions / clk / SM x 148 SMs x 1965 MHz = 18.61 T instr/s nominal.
FP64_INSTR_PER_CLK_SM, N_SM, SM_MAX_MHZ = 64, 148, 1965.0
COUNTERS_CSV = os.path.join(ROOT, "profiles", "r03_step_kernel_counters.csv")


def kernel_rev(version_string):
    """'... kernels r2.1)' -> 'r2.1': the revision tag the ncu counters in profiles/ are recorded against."""
    import re
    m = re.search(r"kernels ([^\s)]+)\)", version_string)
    return m.group(1) if m else None


def load_counters(path=COUNTERS_CSV):
    """workload -> {kernel_rev, fp64_instr_per_cell, dram_bytes_per_launch, source}: per-cell fp64 thread-instructions
    (DADD+DMUL+DFMA+DSETP warp instructions x 32 / cells, halo recomputation included) and dram__bytes_read.sum +
    dram__bytes_write.sum per step-kernel launch, from the committed `ncu --set full` captures."""
    import csv
    out = {}
    try:
        with open(path) as fh:
            for row in csv.DictReader(r for r in fh if not r.startswith("#")):
                out[row["workload"]] = {"kernel_rev": row["kernel_rev"], "fp64_instr_per_cell": float(row["fp64_instr_per_cell"]),
                                        "dram_bytes_per_launch": float(row["dram_bytes_per_launch"]), "source": row["source"]}
    except OSError:
        pass
    return out


def counters_for(workload, version_string, table=None):
    """The counters of `workload` if they were captured for the loaded library's kernel revision, else None (stale)."""
    c = (load_counters() if table is None else table).get(workload)
    if c is None or c["kernel_rev"] != kernel_rev(version_string):
        return None
    return c


def max_over_ranks(x, dist=None, device=None):
    """Time-like quantities are reduced with MAX over ranks (one all-reduce of one double, outside the timed region)."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world, ncell, steps, seconds):
    """Replicas only: every rank advances its own copy of the workload; the job's throughput is the
    cells all ranks updated divided by the slowest rank's time."""
    return world * ncell * steps / seconds


def fp64_roofline(counters, ncell, kern_ms, peak=None, peak_source=None):
    """The viscous 3D step is fp64-ALU-bound before it is HBM-bound: second roofline object.
    counters: counters_for(...) or None; peak in 1e12 fp64 thread-instructions/s (measured) or None (nominal)."""
    if counters is None:
        return None
    if peak is None:
        peak = FP64_INSTR_PER_CLK_SM * N_SM * SM_MAX_MHZ * 1e6 / 1e12
        peak_source = "nominal: 64 fp64 instr/clk/SM x 148 SMs x 1965 MHz"
    ipc = counters["fp64_instr_per_cell"]
    achieved = ipc * ncell / (kern_ms * 1e-3) / 1e12
    return {"bound": "alu", "kernel": "ark_k_step3", "achieved": achieved, "peak": peak, "unit": "T fp64-instr/s",
            "frac": achieved / peak, "fp64_instr_per_cell": ipc, "peak_source": peak_source,
            "counters_from": counters["source"], "kernel_rev": counters["kernel_rev"]}


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def host_cpu():
    """(logical CPUs of the box, CPU model string) for the cpu_baseline record."""
    model = None
    try:
        with open("/proc/cpuinfo") as fh:
            for ln in fh:
                if ln.lower().startswith("model name"):
                    model = ln.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    return os.cpu_count(), model


def oracle_timed(name, steps, warmup):
    """The oracle as it stands, single thread, on a bounded sample of the workload (same recipe, smaller grid)."""
    from oracle import ark_oracle as O
    prm, U, bpc = build_workload(name, device=None, sample=True)
    ncell = prm["nx"] * prm["ny"] * prm["nz"]
    S = U
    for _ in range(warmup):
        S, _ = O.run(prm, S, 1, cfl=CFL)
        S = [S[0], S[1], S[2], S[3] if prm["nz"] > 1 else None, S[4]]
    t0 = time.perf_counter()
    for _ in range(steps):
        S, _ = O.run(prm, S, 1, cfl=CFL)            # compute_dt + step, like the GPU loop
        S = [S[0], S[1], S[2], S[3] if prm["nz"] > 1 else None, S[4]]
    el = time.perf_counter() - t0
    sample = "%s recipe at %dx%dx%d, %d steps of {compute_dt; step}, 1 thread" % (name, prm["nx"], prm["ny"], prm["nz"], steps)
    return ncell * steps / el, el / steps * 1e3, sample


def cpu_baseline_record(val, sample):
    nproc, model = host_cpu()
    return {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, "host_nproc": nproc, "host_cpu": model}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    k = max(1, min(args.steps, 4))
    val, ms, sample = oracle_timed(args.workload, k, 0)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": k,
            "warmup": 0, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "note": "oracle (oracle/ark_oracle.cpp) on host cores; each step is a bounded sample: " + sample},
            "cpu_baseline": cpu_baseline_record(val, sample),
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def measure_workload(name, K, W, dev, local, world, dist, e2e=True, run_steps=0):
    """K timed steps of {compute_dt; step} of one workload (after W warm-up steps), device-timed on the solver's
    stream, max over ranks; the step kernel's own time from events the library records around its launches; optionally
    the end-to-end variant with HOST buffers.  Returns a dict of raw numbers."""
    import torch
    from paper_1903_09043_b200 import binding

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    prm, U, bpc = build_workload(name, device=dev)
    U = [None if a is None else a.reshape(-1).contiguous() for a in U]
    ncell = prm["nx"] * prm["ny"] * prm["nz"]
    s = binding.Solver(prm, device=dev)
    gen = prm.get("phi") is not None
    prm = {k: v for k, v in prm.items() if k != "phi"}      # (the solver holds its padded copy; drop the dense one)
    s.set_state(U)
    for _ in range(W):
        s.step(s.compute_dt(CFL))
    torch.cuda.synchronize()

    # ---- timed region: K x {compute_dt; step}, device-timed on the solver's (= torch current) stream
    s.step_kernel_timing(True)
    l0 = s.launch_count()
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(K):
        s.step(s.compute_dt(CFL))
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms_total = e0.elapsed_time(e1)
    kern_ms, kern_n = s.step_kernel_time()
    s.step_kernel_timing(False)
    launches = s.launch_count() - l0
    ms_total = max_over_ranks(ms_total, dist, dev)
    visc = prm["mu"] > 0 or prm["kappa"] > 0
    out = {"variant": "<VISC=%d,GXY=%d,GEN=%d>" % (visc, gen or prm["g"][0] != 0 or prm["g"][1] != 0, gen) if prm["nz"] > 1
                      else "<2,VISC=%d,GEN=%d>" % (visc, gen),
           "prm": prm, "bpc": bpc, "ncell": ncell, "ms_total": ms_total, "kern_ms": kern_ms, "kern_n": kern_n,
           "launches": launches, "clocks": clocks, "value": whole_job_value(world, ncell, K, ms_total * 1e-3)}

    # sanity: state still finite after the timed steps
    assert s.compute_dt(CFL) > 0

    if run_steps > 0:
        # ---- the same steps through ark_run: dt stays on the device, pairs of steps replayed from a CUDA graph (the 2D
        # configs are launch-latency-bound; this is the loop a user of the library would run)
        s.run(8, CFL)
        l1 = s.launch_count()
        barrier()
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record()
        s.run(run_steps, CFL)
        r1.record()
        barrier()
        run_ms = max_over_ranks(r0.elapsed_time(r1), dist, dev)
        out["ark_run"] = {"steps": run_steps, "us_per_step": run_ms / run_steps * 1e3, "value": whole_job_value(world, ncell, run_steps, run_ms * 1e-3),
                          "unit": UNIT, "gpu_launches": s.launch_count() - l1}

    if e2e:
        # ---- end to end through the C ABI with HOST buffers (pinned): set_state_host + compute_dt + step + get_state_host
        e2e_steps = max(1, min(K, 3))
        host_in = [None if a is None else a.cpu().pin_memory() for a in U]
        host_out = [None if a is None else torch.empty_like(a) .pin_memory() for a in host_in]
        nfield = sum(a is not None for a in host_in)
        s.set_state_host(host_in)
        s.step(s.compute_dt(CFL))
        s.get_state_host(host_out)                      # warm-up of the e2e path
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            s.set_state_host(host_in)
            s.step(s.compute_dt(CFL))
            s.get_state_host(host_out)
        torch.cuda.synchronize()
        e2e_s = max_over_ranks(time.perf_counter() - t0, dist, dev)
        out["e2e"] = {"value": whole_job_value(world, ncell, e2e_steps, e2e_s), "unit": UNIT,
                      "h2d_bytes_per_step": nfield * ncell * 8, "d2h_bytes_per_step": nfield * ncell * 8 + 16, "steps": e2e_steps,
                      "path": "ark_set_state_host + ark_compute_dt + ark_step + ark_get_state_host, pinned host buffers"}
    s.close()
    del s, U
    torch.cuda.empty_cache()
    return out


def measure_slab(name, K, W, dev, local, world, rank, dist):
    """Opt-in `--decomp slab`: ONE global workload split along z over the ranks
    (strong scaling), halo planes exchanged before every step (NCCL P2P over NVLink), dt = min over ranks.  Device-timed,
    max over ranks; value = global cells * K / time."""
    import torch
    from paper_1903_09043_b200 import binding, inputs, slab
    fn, n, bpc, _ = WORKLOADS[name]
    k0, k1 = slab.partition(n, world)[rank]
    prm, U = getattr(inputs, fn)(n, device=dev, box=((k0, k1), (0, n), (0, n)))
    U = [a.reshape(-1).contiguous() for a in U]
    s = slab.SlabSolver(binding, prm, rank, world, dist if world > 1 else None, device=dev)
    s.set_state(U)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(W):
        s.step(s.compute_dt(CFL))
    l0 = s.s.launch_count()
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(K):
        s.step(s.compute_dt(CFL))
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms_total = max_over_ranks(e0.elapsed_time(e1), dist, dev)
    launches = s.s.launch_count() - l0
    assert s.compute_dt(CFL) > 0
    out = {"ncell": n ** 3, "bpc": bpc, "ms_total": ms_total, "launches": launches, "clocks": clocks,
           "value": n ** 3 * K / (ms_total * 1e-3), "halo_bytes_sent_per_step_per_rank": s.bytes_per_exchange(),
           "planes": [k0, k1], "grid": [n, n, n]}
    s.close()
    return out


def roofline_objects(name, m, world, version, fp64_peak):
    """(hbm roofline, fp64 roofline) of one measured workload."""
    peak, peak_src = measured_peaks()
    alg_bytes = m["bpc"] * m["ncell"]                 # per launch of the dominant (fused step) kernel
    kern_avg_ms = m["kern_ms"] / max(m["kern_n"], 1)
    achieved = alg_bytes / (kern_avg_ms * 1e-3) / 1e9
    c = counters_for(name, version)
    hbm = {"bound": "hbm", "kernel": ("ark_k_step3" if m["prm"]["nz"] > 1 else "ark_k_step") + m["variant"], "achieved": achieved, "peak": peak, "unit": "GB/s",
           "frac": achieved / peak, "traffic": c["dram_bytes_per_launch"] if c else None,
           "traffic_from": c["source"] if c else "no ncu capture of kernel revision %s in profiles/" % kernel_rev(version),
           "peak_source": peak_src, "algorithmic_bytes_per_cell": m["bpc"], "kernel_ms": kern_avg_ms,
           "kernel_launches_timed": m["kern_n"], "kernel_share_of_step": m["kern_ms"] / m["ms_total"],
           "effective_whole_step_frac": m["bpc"] * m["value"] / world / 1e9 / peak}
    alu = fp64_roofline(c, m["ncell"], kern_avg_ms, fp64_peak,
                        "measured in this run (ark_measure_fp64_peak: register-resident DFMA chains; nominal 18.61)" if fp64_peak else None)
    return hbm, alu


def run_ours(args):
    import torch
    from paper_1903_09043_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    binding.load()
    version = binding.version_string()
    W = max(args.warmup, 3)
    K = args.steps
    if args.decomp == "slab":
        m = measure_slab(args.workload, K, W, dev, local, world, rank, dist)
        if rank == 0:
            peak, peak_src = measured_peaks()
            print(json.dumps({
                "metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": m["ms_total"] / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": args.workload, "grid": m["grid"], "cfl": CFL, "parallelism": "slab decomposition along z, %d ranks" % world,
                           "step": "min-all-reduce of dt + halo exchange (2 planes x 5 fields per neighbour, NCCL P2P) + ark_step per rank",
                           "l2": "inputs larger than L2", "library": version},
                "roofline": {"bound": "hbm", "kernel": "ark_k_step3", "achieved": m["bpc"] * m["value"] / world / 1e9, "peak": peak, "unit": "GB/s",
                             "frac": m["bpc"] * m["value"] / world / 1e9 / peak, "traffic": None, "peak_source": peak_src,
                             "note": "whole-step effective algorithmic bandwidth per GPU (exchange included)"},
                "halo_bytes_sent_per_step_per_rank": m["halo_bytes_sent_per_step_per_rank"],
                "gpu_launches": m["launches"], "clocks": m["clocks"]}))
        if dist is not None:
            dist.destroy_process_group()
        return
    m = measure_workload(args.workload, K, W, dev, local, world, dist, e2e=not args.no_e2e)
    fp64_peak = binding.measure_fp64_peak()
    also = []
    if args.workload == "config5_512" and not args.no_also:
        # the other roofline target of north_star (config4_256), the kernel variants no BASELINE config selects and the
        # three 2D BASELINE configs: same measurement, same driver-run line, each with its own clocks record
        for name2, k2, run2 in ALSO:
            also.append((name2, measure_workload(name2, k2, W, dev, local, world, dist, e2e=False, run_steps=run2)))

    if rank == 0:
        prm, bpc, ncell = m["prm"], m["bpc"], m["ncell"]
        hbm, alu = roofline_objects(args.workload, m, world, version, fp64_peak)
        line = {"metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": m["ms_total"] / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": args.workload, "grid": [prm["nx"], prm["ny"], prm["nz"]], "cfl": CFL,
                           "step": "ark_compute_dt + ark_step (ghost fill y/z, fused step kernel incl. periodic x ghosts, CFL pass 2, 16 B D2H)",
                           "l2": "inputs larger than L2 (state %.2f GB)" % (bpc / 2 * ncell / 1e9) if bpc / 2 * ncell > 200e6
                                 else "state fits in L2 (%.1f MB): latency-bound config, HBM roofline not meaningful" % (bpc / 2 * ncell / 1e6),
                           "parallelism": "replicas only" if world > 1 else "single GPU",
                           "library": version},
                "roofline": hbm, "roofline_fp64": alu, "e2e": m.get("e2e"), "gpu_launches": m["launches"], "clocks": m["clocks"]}
        if also:
            line["also"] = []
            for name2, m2 in also:
                hbm2, alu2 = roofline_objects(name2, m2, world, version, fp64_peak)
                k2 = m2["kern_n"]
                ent = {"workload": name2, "grid": [m2["prm"]["nx"], m2["prm"]["ny"], m2["prm"]["nz"]], "steps": k2,
                       "value": m2["value"], "unit": UNIT, "ms_per_step": m2["ms_total"] / k2, "roofline": hbm2,
                       "roofline_fp64": alu2, "gpu_launches": m2["launches"], "clocks": m2["clocks"]}
                if "ark_run" in m2:
                    ent["ark_run"] = m2["ark_run"]
                line["also"].append(ent)
        if world == 1 and not args.no_cpu_baseline:
            val, ms, sample = oracle_timed(args.workload, 2, 0)
            line["cpu_baseline"] = cpu_baseline_record(val, sample)
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def spawn_ranks(args):
    """`python bench.py --gpus N` without a torchrun environment: re-launch under torch.distributed.run, one rank per GPU
    (the launch line the driver itself uses), and pass its output through."""
    import socket
    sk = socket.socket()
    sk.bind(("127.0.0.1", 0))
    port = sk.getsockname()[1]
    sk.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config5_512", choices=sorted(WORKLOADS))
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default, north_star: the path does not shard) or ONE workload split along z (slab.py)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg (kernel tuning runs)")
    ap.add_argument("--no-also", action="store_true", help="skip the other workloads that ride along with config5_512")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args))
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
