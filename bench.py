#!/usr/bin/env python
"""bench.py -- particle-steps/s of the forward + adjoint PM hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference]

One "step" is one pass of the whole hot path: pm_run_fwd_adj on one batch of seeded synthetic input
(acc_0, n KDK steps forward, objective, n adjoint steps with reverse-time integration; SURVEY.md §8a
rows a1-a19).  value = N_p * n * K / time  [particle-steps/s, forward + adjoint counted once].
N > 1 (torchrun): the path does not shard; every rank runs an
independent replica on its own seed, no collective in the data path, value = sum over ranks / max time.
--impl reference times the CPU fp64 ORACLE (oracle/) on a bounded sample of the same workload.
Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
from paper_2211_09815_b200 import inputs  # noqa: E402  (seeded generators only; no arithmetic of the method)

METRIC = "particle-steps/s (fwd+adjoint)"
UNIT = "particle-steps/s"


def make_inputs(k, p_over_s, seed_offset=0):
    cfg = inputs.config(k)
    s0 = inputs.zeldovich_displacement(cfg["lattice"], cfg["mesh"], seed=1 + 100 * seed_offset, rms=0.3)
    p0 = (s0.astype(np.float64) * p_over_s(cfg)).astype(np.float32)
    target = inputs.lognormal_target(cfg["mesh"], seed=2 + 100 * seed_offset, sigma=1.0)
    return cfg, s0, p0, target


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([v.strip() for v in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 7 and r[3 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def max_over_ranks(ms, world, device):
    """Replicas: the job's time is the slowest rank's device time."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(world, npart, n_steps, runs, ms):
    """Whole-job particle-steps/s: every rank runs its own replica of the same size, no data-path collective."""
    return world * npart * n_steps * runs / (ms * 1e-3)


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def oracle_sample(cfg, s0, p0, target, n_sample):
    """Times the oracle, as it stands, on the first n_sample KDK steps forward + the matching adjoint steps."""
    from oracle import pm_oracle as orc
    orc.build()
    a = cfg["a"][: n_sample + 1]
    t = time.perf_counter()
    orc.run_fwd_adj(cfg["mesh"], cfg["lattice"], cfg["omega_m"], a, s0, p0, target)
    dt = time.perf_counter() - t
    npart = s0.shape[0]
    return npart * n_sample / dt, dt, orc.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import pm_oracle as orc
    orc.build()
    cfg, s0, p0, target = make_inputs(args.config, lambda c: orc.p_over_s(c["omega_m"], c["a"][0]))
    n_sample = args.ref_steps
    vals = []
    for it in range(args.warmup + args.steps):
        v, dt, threads = oracle_sample(cfg, s0, p0, target, n_sample)
        if it >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([dt for _, dt in vals]) * 1e3)
    sample = f"first {n_sample} of {cfg['n_steps']} KDK steps forward + adjoint (incl. acc_0 and objective) at full size"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "particles": int(s0.shape[0]), "mesh": list(cfg["mesh"]), "kdk_steps": n_sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2211_09815_b200 import binding  # raises if libpm.so is missing: no fallback

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def p_over_s(c):
        g = binding.host_growth(c["omega_m"], c["a"][0])
        return g[2] / g[0]

    cfg, s0, p0, target = make_inputs(args.config, p_over_s, seed_offset=rank)
    n, npart = cfg["n_steps"], s0.shape[0]
    pm = binding.PM(cfg["mesh"], cfg["lattice"], cfg["omega_m"], cfg["a"], device=f"cuda:{local}")
    s0d, p0d, tgd = (torch.from_numpy(v).cuda() for v in (s0, p0, target))
    outs = {k: torch.empty((npart, 3), dtype=torch.float32, device="cuda") for k in ("s_n", "p_n", "xi0", "pi0", "dJ_ds0")}
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed(fn, steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        for _ in range(steps):
            fn()
        e1.record(stream)
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), world, "cuda")

    J = [0.0]

    def step_dev():
        J[0] = pm.run_fwd_adj(s0d, p0d, tgd, out=outs)["J"]

    # ---- device-resident timing (value): K steps, nothing but the run in the timed region ----
    for _ in range(args.warmup):
        step_dev()
    own0, fft0 = pm.launch_count()
    clocks = ClockSampler(local)
    ms = timed(step_dev, args.steps)
    clk = clocks.stop()
    own1, fft1 = pm.launch_count()
    value = job_value(world, npart, n, args.steps, ms)

    # ---- the same K steps again with a CUDA-event pair around every launch (recorded by libpm on its own stream):
    #      per-kernel durations for the roofline and the kernel table.  The events cost a few per cent of the step
    #      (ms_per_step_instrumented), which is why `value` is not taken from this pass. ----
    tm = {}
    ms_instr = None
    if not args.no_kernel_timing:
        pm.timing_enable(True)
        pm.timing_reset()
        ms_instr = timed(step_dev, args.steps)
        tm = pm.timing_read()
        pm.timing_enable(False)
        pm.timing_reset()

    # ---- end to end through host buffers (e2e): H2D of inputs and D2H of results inside the timed region ----
    hin = [torch.from_numpy(v).pin_memory() for v in (s0, p0, target)]
    hout = {k: torch.empty((npart, 3), dtype=torch.float32).pin_memory() for k in ("s_n", "p_n", "dJ_ds0")}

    def step_host():
        J[0] = pm.run_fwd_adj_host(hin[0], hin[1], hin[2], hout)

    step_host()
    ms_h = timed(step_host, args.steps)
    e2e = job_value(world, npart, n, args.steps, ms_h)
    h2d = sum(t.numel() * 4 for t in hin)
    d2h = sum(t.numel() * 4 for t in hout.values()) + 8

    # ---- roofline of the dominant own kernel + the per-kernel table ----
    peak, peak_src = measured_peak_gbs()
    kernels = {}
    tot_ms = sum(v["ms"] for v in tm.values()) or 1.0
    for name, v in tm.items():
        if v["launches"]:
            per_ms = v["ms"] / v["launches"]
            gbs = v["algo_bytes"] / v["launches"] / (per_ms * 1e-3) / 1e9
            kernels[name] = {"launches_per_step": v["launches"] / args.steps, "avg_ms": per_ms, "share": v["ms"] / tot_ms,
                             "algo_GBps": gbs, "frac_of_peak": gbs / peak}
    own = {k: v for k, v in kernels.items() if k not in ("fft_r2c", "fft_c2r")}  # cuFFT calls are listed, not graded
    if not own:  # --no-kernel-timing
        own = {"none": {"share": 0.0, "algo_GBps": 0.0}}
    dom = max(own, key=lambda k: own[k]["share"])
    traffic = None  # DRAM bytes per launch of that kernel from the committed ncu --set full capture (profiles/), or null
    try:
        with open(os.path.join(ROOT, "profiles", "r01b_traffic.csv")) as f:
            for ln in f:
                parts = ln.strip().split(",")
                if len(parts) == 3 and parts[0] == cfg["name"] and parts[1] == dom:
                    traffic = float(parts[2])
    except Exception:
        pass
    roofline = {"bound": "hbm", "kernel": dom, "achieved": own[dom]["algo_GBps"], "peak": peak, "unit": "GB/s",
                "frac": own[dom]["algo_GBps"] / peak, "traffic": traffic, "peak_source": peak_src,
                "share_of_step": own[dom]["share"],
                "timing": "CUDA events around every launch on the library's stream, second pass of the same K steps"}

    line = None
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": {"workload": cfg["name"], "particles": int(npart), "mesh": list(cfg["mesh"]), "kdk_steps": n,
                           "omega_m": cfg["omega_m"], "parallelism": "replicas" if world > 1 else "single",
                           "l2": "working set (%.2f GB workspace) larger than the 126 MB L2" % (pm.workspace_nbytes / 1e9)},
                "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "ms_per_step": ms_h / args.steps},
                "gpu_launches": int(own1 - own0), "cufft_calls": int(fft1 - fft0),
                "ms_per_step_instrumented": None if ms_instr is None else ms_instr / args.steps,
                "clocks": clk, "roofline": roofline, "kernels": kernels, "objective_J": J[0],
                "peak_mem_GB": torch.cuda.max_memory_allocated() / 1e9}
        if world == 1 and not args.no_cpu_baseline:
            v, dt, threads = oracle_sample(cfg, s0, p0, target, args.ref_steps)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "seconds": dt,
                                    "sample": f"first {args.ref_steps} of {n} KDK steps forward + adjoint at full size "
                                              f"({cfg['name']})"}
        print(json.dumps(line), flush=True)
    pm.close()
    if world > 1:
        dist.destroy_process_group()


def run_sweep(args):
    """configs[4]: CIC scatter / gather / weight-gradient gather of 512^3 particles on a 1024^3 mesh, clustered
    (20000 Gaussian blobs, 70 % of the particles) against uniform positions, in generation and in random memory
    order; GB/s = SURVEY section 8d algorithmic bytes / CUDA-event time, with and without the binning pass."""
    import torch
    from paper_2211_09815_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(0)
    L = args.sweep_lattice
    N = 2 * L
    mesh, npart = (N, N, N), L ** 3
    pm = binding.PM(mesh, (L, L, L), 0.3, [1.0])
    peak, peak_src = measured_peak_gbs()
    gen = torch.Generator(device="cuda").manual_seed(5)
    f3 = torch.randn((3,) + mesh, device="cuda", generator=gen)
    val = torch.randn((npart, 3), device="cuda", generator=gen)
    ng = float(N) ** 3
    algo = {"scatter1": 12.0 * npart + 4.0 * ng, "scatter3": 24.0 * npart + 12.0 * ng, "gather3": 24.0 * npart + 12.0 * ng,
            "gather_grad1": 24.0 * npart + 4.0 * ng}
    ops = {"scatter1": lambda x: pm.scatter(x), "scatter3": lambda x: pm.scatter(x, val), "gather3": lambda x: pm.gather(x, f3),
           "gather_grad1": lambda x: pm.gather_grad(x, f3[0])}
    cls_of = {"scatter1": "scatter1", "scatter3": "scatter3", "gather3": "gather", "gather_grad1": "gather_grad"}
    n_blobs = max(1, int(round(20000 * npart / 512.0 ** 3)))
    cases = {"clustered/generation": lambda: inputs.blob_positions(npart, mesh, seed=3, n_blobs=n_blobs, order="generation"),
             "clustered/random": lambda: inputs.blob_positions(npart, mesh, seed=3, n_blobs=n_blobs, order="random"),
             "uniform/generation": lambda: inputs.uniform_positions(npart, mesh, seed=3)}
    out = {}
    for cname, make in cases.items():
        x = torch.from_numpy(make()).cuda()
        res = {}
        for oname, op in ops.items():
            for _ in range(max(args.warmup, 1)):
                op(x)
            torch.cuda.synchronize()
            pm.timing_enable(True)
            pm.timing_reset()
            for _ in range(args.steps):
                op(x)
            torch.cuda.synchronize()
            tm = pm.timing_read()
            pm.timing_enable(False)
            pm.timing_reset()
            k_ms = tm[cls_of[oname]]["ms"] / args.steps
            bin_ms = sum(tm[b]["ms"] for b in ("bin_count", "bin_scan", "bin_reorder")) / args.steps
            res[oname] = {"kernel_ms": k_ms, "binning_ms": bin_ms, "GBps": algo[oname] / (k_ms * 1e-3) / 1e9,
                          "frac_of_peak": algo[oname] / (k_ms * 1e-3) / 1e9 / peak,
                          "GBps_with_binning": algo[oname] / ((k_ms + bin_ms) * 1e-3) / 1e9}
        out[cname] = res
        del x
    line = {"metric": "CIC scatter/gather GB/s vs HBM peak (kernel sweep)", "value": out["clustered/generation"]["scatter1"]["GBps"],
            "unit": "GB/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "higher_is_better": True, "dtype": "f32",
            "data": "synthetic", "vs_baseline": None,
            "config": {"workload": f"cfg4_kernel_sweep_{L}p_{N}m", "particles": npart, "mesh": list(mesh), "blobs": n_blobs},
            "peak": peak, "peak_source": peak_src, "sweep": out, "peak_mem_GB": torch.cuda.max_memory_allocated() / 1e9}
    print(json.dumps(line), flush=True)
    pm.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index (0-3; 4 = the CIC kernel sweep)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-steps", type=int, default=1, help="KDK steps in the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-kernel-timing", action="store_true", help="no per-kernel CUDA events in the timed region (debug)")
    ap.add_argument("--sweep-lattice", type=int, default=512, help="particles per axis of the configs[4] kernel sweep (mesh = 2x)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.config == 4:
        run_sweep(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
