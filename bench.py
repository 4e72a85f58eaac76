#!/usr/bin/env python
"""bench.py -- particle-steps/s of the forward + adjoint PM hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

One "step" is one pass of the whole hot path: pm_run_fwd_adj on one batch of seeded synthetic input
(acc_0, n KDK steps forward, objective, n adjoint steps with reverse-time integration; SURVEY.md section 8a
rows a1-a19).  value = N_p * n * K / time  [particle-steps/s, forward + adjoint counted once].

Headline workload: configs[2] (256^3 particles, 512^3 mesh, 63 steps) -- the largest config for which BOTH arms
(this one and --impl reference) finish well inside the driver's per-arm limit at --steps 20 --warmup 5 (DESIGN.md
section 9 has the arithmetic).  The same JSON line carries, at N = 1:
  scale_up.cfg3   configs[3] (512^3 / 1024^3, 100 steps): 1 warm-up + 2 runs, kernel table, peak memory, and the
                  peak-memory triple for n = 25, 50, 100 steps (torch peak + cudaMemGetInfo delta);
  sweep.cfg4      configs[4]: CIC scatter / gather / weight-gradient gather of 512^3 particles on a 1024^3 mesh,
                  clustered vs uniform positions, generation vs random memory order, kernel-only and with binning.
  split           forward-only and adjoint-only rates of the headline workload (step-by-step ABI calls);
  modes           the headline workload in the fp64-transform mode (pm_params.flags, the mode that meets the 1e-3 gradient bar);
  next_rows       milliseconds per call of the SURVEY 8f rows (device ICs and their VJP, observed snapshots, dJ/dOmega_m, Adam).
N > 1 (torchrun): the path does not shard; every rank runs an independent
replica on its own seed, no collective in the data path, value = sum over ranks / max time.
--impl reference times the CPU fp64 ORACLE (oracle/) on bounded samples of the same workload.
Prints ONE JSON line on rank 0.
"""
import argparse
import hashlib
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
GRADED = ("scatter1", "scatter3", "gather", "gather_grad", "gather_fused", "gather_kick", "kspace_force", "kspace_adjoint")
T_START = time.time()


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


class FreeMemSampler:
    """Lowest cudaMemGetInfo 'free' seen while a run is in flight (cuFFT's own allocations are invisible to torch)."""

    def __init__(self, torch, device, period=0.05):
        self.torch, self.device, self.period = torch, device, period
        self.min_free = torch.cuda.mem_get_info(device)[0]
        self._stop = threading.Event()
        self.th = threading.Thread(target=self._run, daemon=True)
        self.th.start()

    def _run(self):
        while not self._stop.is_set():
            self.min_free = min(self.min_free, self.torch.cuda.mem_get_info(self.device)[0])
            time.sleep(self.period)

    def stop(self):
        self._stop.set()
        self.th.join()
        self.min_free = min(self.min_free, self.torch.cuda.mem_get_info(self.device)[0])
        return self.min_free


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


def source_hash():
    """sha256 over the kernel sources: ties a committed ncu traffic figure to the code it was captured from."""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2211_09815_b200", "csrc")
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh", ".inc")):
            with open(os.path.join(d, name), "rb") as f:
                h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def committed_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed ncu --set full capture of this
    workload (profiles/r02_traffic.csv: workload,kernel,bytes_per_launch,source_hash,commit), or None when there is no row
    or the row was captured from other kernel sources than the ones running now."""
    try:
        with open(os.path.join(ROOT, "profiles", "r02_traffic.csv")) as f:
            rows = [ln.strip().split(",") for ln in f if ln.strip() and not ln.startswith("#")]
    except OSError:
        return None, "no profiles/r02_traffic.csv"
    cur = source_hash()
    for r in rows:
        if len(r) >= 5 and r[0] == workload and r[1] == kernel:
            if r[3] != cur:
                return None, f"capture of commit {r[4]} (sources {r[3]}) predates the running sources ({cur})"
            return float(r[2]), f"ncu --set full at commit {r[4]}"
    return None, "no capture for this workload / kernel"


# ---- the oracle, timed on the host cores ---------------------------------------------------------------------------------
def oracle_steady_sample(cfg, s0, p0, target, n_pairs):
    """Times the oracle, as it stands, on n_pairs forward KDK steps and n_pairs adjoint steps in steady state at full
    size.  acc_0 = F(x_0) and the objective (which every run pays once, not once per step) are executed but NOT billed,
    so the figure is the per-step cost the GPU's particle-steps/s is compared with: 1 force evaluation per forward step,
    1 force + 1 force VJP per adjoint step."""
    from oracle import pm_oracle as orc
    orc.build()
    N, L, om, a = cfg["mesh"], cfg["lattice"], cfg["omega_m"], cfg["a"]
    s = np.ascontiguousarray(s0, dtype=np.float64).copy()
    p = np.ascontiguousarray(p0, dtype=np.float64).copy()
    acc = orc.init_acc(N, L, om, s)
    t0 = time.perf_counter()
    for i in range(1, n_pairs + 1):
        orc.step_fwd(N, L, om, a, i, s, p, acc)
    t_fwd = time.perf_counter() - t0
    _, xi = orc.objective(N, orc.positions(N, L, s), target)
    pi = np.zeros_like(s)
    alpha = np.zeros_like(s)
    t0 = time.perf_counter()
    for i in range(n_pairs, 0, -1):
        orc.step_adj(N, L, om, a, i, s, p, acc, xi, pi, alpha)
    t_adj = time.perf_counter() - t0
    return s0.shape[0] * n_pairs / (t_fwd + t_adj), t_fwd, t_adj, orc.num_threads()


def sample_text(cfg, n_pairs):
    return (f"{n_pairs} forward + {n_pairs} adjoint KDK steps in steady state at full size ({cfg['name']}); "
            "acc_0 and the objective executed, not billed")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import pm_oracle as orc
    orc.build()
    cfg, s0, p0, target = make_inputs(args.config, lambda c: orc.p_over_s(c["omega_m"], c["a"][0]))
    n_pairs = max(1, args.ref_steps)
    vals, t_used, warm_done = [], 0.0, 0
    want_warm = min(args.warmup, 1)  # a CPU program has nothing to warm but its page faults: one untimed sample at most
    while len(vals) < args.steps:
        t0 = time.perf_counter()
        v, tf, ta, threads = oracle_steady_sample(cfg, s0, p0, target, n_pairs)
        dt_total = time.perf_counter() - t0
        t_used += dt_total
        if warm_done < want_warm:
            warm_done += 1
        else:
            vals.append((v, tf + ta))
        # bounded: never start a sample that would push the arm beyond its budget (at least 2 samples are timed)
        if len(vals) >= 2 and t_used + dt_total > args.ref_budget_s:
            break
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([dt for _, dt in vals]) * 1e3)
    sample = sample_text(cfg, n_pairs)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": len(vals),
            "steps_requested": args.steps, "warmup": warm_done, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "particles": int(s0.shape[0]), "mesh": list(cfg["mesh"]), "kdk_steps": cfg["n_steps"],
                       "omega_m": cfg["omega_m"], "parallelism": "single"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "budget_s": args.ref_budget_s}
    print(json.dumps(line), flush=True)


# ---- kernel table helpers --------------------------------------------------------------------------------------------------
def kernel_table(tm, steps, peak):
    kernels = {}
    tot_ms = sum(v["ms"] for v in tm.values()) or 1.0
    for name, v in tm.items():
        if v["launches"]:
            per_ms = v["ms"] / v["launches"]
            gbs = v["algo_bytes"] / v["launches"] / (per_ms * 1e-3) / 1e9
            kernels[name] = {"launches_per_step": v["launches"] / steps, "avg_ms": per_ms, "share": v["ms"] / tot_ms,
                             "algo_bytes_per_launch": v["algo_bytes"] / v["launches"], "algo_GBps": gbs, "frac_of_peak": gbs / peak}
    return kernels


def graded_roofline(kernels, workload, peak, peak_src):
    """roofline of the dominant GRADED kernel (north_star: CIC scatter / gather and k-space classes; the transform passes
    are listed in `kernels`, not graded)."""
    graded = {k: v for k, v in kernels.items() if k in GRADED}
    if not graded:
        return {"bound": "hbm", "kernel": None, "achieved": 0.0, "peak": peak, "unit": "GB/s", "frac": 0.0, "traffic": None,
                "peak_source": peak_src}
    dom = max(graded, key=lambda k: graded[k]["share"])
    traffic, note = committed_traffic(workload, dom)
    return {"bound": "hbm", "kernel": dom, "achieved": graded[dom]["algo_GBps"], "peak": peak, "unit": "GB/s",
            "frac": graded[dom]["algo_GBps"] / peak, "traffic": traffic, "traffic_source": note, "peak_source": peak_src,
            "algo_bytes_per_launch": graded[dom]["algo_bytes_per_launch"], "avg_ms": graded[dom]["avg_ms"],
            "share_of_step": graded[dom]["share"],
            "graded_fracs": {k: round(v["frac_of_peak"], 4) for k, v in graded.items()},
            "timing": "CUDA events around every launch on the library's stream, second pass of the same K steps"}


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
    device = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
    peak, peak_src = measured_peak_gbs()

    def p_over_s(c):
        g = binding.host_growth(c["omega_m"], c["a"][0])
        return g[2] / g[0]

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    stream = torch.cuda.current_stream()

    def timed(fn, steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        for _ in range(steps):
            fn()
        e1.record(stream)
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), world, "cuda")

    # ================= headline =================
    cfg, s0, p0, target = make_inputs(args.config, p_over_s, seed_offset=rank)
    n, npart = cfg["n_steps"], s0.shape[0]
    pm = binding.PM(cfg["mesh"], cfg["lattice"], cfg["omega_m"], cfg["a"], device=f"cuda:{local}")
    s0d, p0d, tgd = (torch.from_numpy(v).cuda() for v in (s0, p0, target))
    outs = {k: torch.empty((npart, 3), dtype=torch.float32, device="cuda") for k in ("s_n", "p_n", "xi0", "pi0", "dJ_ds0")}
    J = [0.0]

    def step_dev():
        J[0] = pm.run_fwd_adj(s0d, p0d, tgd, out=outs)["J"]

    for _ in range(args.warmup):
        step_dev()
    own0, fft0 = pm.launch_count()
    clocks = ClockSampler(local)
    ms = timed(step_dev, args.steps)
    clk = clocks.stop()
    own1, fft1 = pm.launch_count()
    value = job_value(world, npart, n, args.steps, ms)

    # the same K steps again with a CUDA-event pair around every launch (recorded by libpm on its own stream): per-kernel
    # durations for the roofline and the kernel table.  The events (and the serialisation of the two adjoint branches
    # they force) cost a few per cent of the step, which is why `value` is not taken from this pass.
    kernels, ms_instr = {}, None
    if not args.no_kernel_timing:
        pm.timing_enable(True)
        pm.timing_reset()
        ms_instr = timed(step_dev, args.steps)
        kernels = kernel_table(pm.timing_read(), args.steps, peak)
        pm.timing_enable(False)
        pm.timing_reset()

    # forward-only and adjoint-only rates through the step-by-step ABI calls (pm_set_state + n pm_step_fwd;
    # pm_objective + n pm_step_adj): the same kernels as the whole run without the chaining of kick / drift across steps
    split = None
    if world == 1 and not args.no_kernel_timing:
        def fwd_only():
            pm.set_state(s0d, p0d)
            for i in range(1, n + 1):
                pm.step_fwd(i)

        def adj_only():
            pm.objective(tgd)
            for i in range(n, 0, -1):
                pm.step_adj(i)

        fwd_only()
        adj_only()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        torch.cuda.synchronize()
        ev[0].record(stream)
        fwd_only()
        ev[1].record(stream)
        adj_only()
        ev[2].record(stream)
        torch.cuda.synchronize()
        tf, ta = ev[0].elapsed_time(ev[1]), ev[1].elapsed_time(ev[2])
        split = {"forward_only": {"value": npart * n / (tf * 1e-3), "unit": UNIT, "ms": tf},
                 "adjoint_only": {"value": npart * n / (ta * 1e-3), "unit": UNIT, "ms": ta},
                 "note": "step-by-step ABI calls (acc_0 billed to the forward part, the objective to the adjoint part), "
                         "1 warm-up + 1 timed pass; the whole run chains kick / drift across steps and is faster than the sum"}

    # end to end through host buffers (e2e): H2D of inputs and D2H of results inside the timed region
    hin = [torch.from_numpy(v).pin_memory() for v in (s0, p0, target)]
    hout = {k: torch.empty((npart, 3), dtype=torch.float32).pin_memory() for k in ("s_n", "p_n", "dJ_ds0")}

    def step_host():
        J[0] = pm.run_fwd_adj_host(hin[0], hin[1], hin[2], hout)

    step_host()
    ms_h = timed(step_host, args.steps)
    e2e = job_value(world, npart, n, args.steps, ms_h)
    h2d = sum(t.numel() * 4 for t in hin)
    d2h = sum(t.numel() * 4 for t in hout.values()) + 8
    peak_mem = torch.cuda.max_memory_allocated() / 1e9
    ws_gb = pm.workspace_nbytes / 1e9
    pm.close()
    del pm, s0d, p0d, tgd, outs, hin, hout
    torch.cuda.empty_cache()

    line = None
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": {"workload": cfg["name"], "particles": int(npart), "mesh": list(cfg["mesh"]), "kdk_steps": n,
                           "omega_m": cfg["omega_m"], "parallelism": "replicas" if world > 1 else "single",
                           "l2": "inputs larger than L2: every kernel streams meshes of %.2f GB each (L2 = 126 MB), no flush needed"
                                 % (4.0 * np.prod(cfg["mesh"]) / 1e9) if np.prod(cfg["mesh"]) * 4 > 3 * 126e6 else
                                 "one mesh (%.0f MB) is smaller than the 126 MB L2: per-kernel fractions at this size are L2-assisted upper bounds"
                                 % (4.0 * np.prod(cfg["mesh"]) / 1e6)},
                "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "ms_per_step": ms_h / args.steps},
                "gpu_launches": int(own1 - own0), "cufft_calls": int(fft1 - fft0),
                "ms_per_step_instrumented": None if ms_instr is None else ms_instr / args.steps,
                "clocks": clk, "roofline": graded_roofline(kernels, cfg["name"], peak, peak_src), "kernels": kernels,
                "objective_J": J[0], "peak_mem_GB": peak_mem, "workspace_GB": ws_gb}
        if split:
            line["split"] = split
        if world == 1 and not args.no_cpu_baseline:
            n_pairs = args.cpu_pairs
            v, tf, ta, threads = oracle_steady_sample(cfg, s0, p0, target, n_pairs)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "seconds": tf + ta,
                                    "seconds_forward": tf, "seconds_adjoint": ta, "sample": sample_text(cfg, n_pairs)}
    del s0, p0, target

    # ================= sub-records (N = 1 only; each guarded, a failure is recorded, not fatal) =================
    if rank == 0 and world == 1 and not args.no_modes:
        try:
            line["modes"] = {"fp64_transforms": mode_fp64_transforms(args, torch, binding, p_over_s)}
        except Exception as e:  # noqa: BLE001
            line["modes"] = {"fp64_transforms": {"error": f"{type(e).__name__}: {e}"}}
        torch.cuda.empty_cache()
        try:
            line["next_rows"] = next_rows_cfg1(torch, binding, p_over_s)
        except Exception as e:  # noqa: BLE001
            line["next_rows"] = {"error": f"{type(e).__name__}: {e}"}
        torch.cuda.empty_cache()
    if rank == 0 and world == 1 and args.config == 2:
        if not args.no_scale_up:
            try:
                line["scale_up"] = {"cfg3": scale_up_cfg3(args, torch, binding, p_over_s, peak, peak_src, local)}
            except Exception as e:  # noqa: BLE001
                line["scale_up"] = {"cfg3": {"error": f"{type(e).__name__}: {e}"}}
            torch.cuda.empty_cache()
        if not args.no_sweep:
            try:
                line["sweep"] = {"cfg4": sweep_cfg4(args, torch, binding, peak, peak_src, args.sweep_lattice)}
            except Exception as e:  # noqa: BLE001
                line["sweep"] = {"cfg4": {"error": f"{type(e).__name__}: {e}"}}
    if rank == 0:
        line["wall_s"] = time.time() - T_START
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def _events_ms(torch, fn, reps=1):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def mode_fp64_transforms(args, torch, binding, p_over_s):
    """The headline workload in the PM_FLAG_FP64_TRANSFORMS mode (transforms and k-space operators in fp64: the mode that
    meets north_star's 1e-3 gradient bar at configs[1], tests/test_gpu_full_size.py): 1 warm-up + 2 timed runs."""
    cfg, s0, p0, target = make_inputs(args.config, p_over_s)
    npart = s0.shape[0]
    pm = binding.PM(cfg["mesh"], cfg["lattice"], cfg["omega_m"], cfg["a"], flags=binding.PM_FLAG_FP64_TRANSFORMS)
    dv = [torch.from_numpy(v).cuda() for v in (s0, p0, target)]
    outs = {k: torch.empty((npart, 3), dtype=torch.float32, device="cuda") for k in ("s_n", "p_n", "xi0", "pi0", "dJ_ds0")}
    J = [0.0]

    def step():
        J[0] = pm.run_fwd_adj(*dv, out=outs)["J"]

    step()
    ms = _events_ms(torch, step, 2)
    rec = {"workload": cfg["name"], "value": npart * cfg["n_steps"] / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "steps": 2,
           "warmup": 1, "workspace_GB": pm.workspace_nbytes / 1e9, "objective_J": J[0],
           "note": "transforms via cuFFT D2Z/Z2D + fp64 k-space kernels; all particle and mesh arrays fp32"}
    pm.close()
    return rec


def next_rows_cfg1(torch, binding, p_over_s):
    """SURVEY 8f rows at configs[1]'s sizes, milliseconds per call (CUDA events, 1 warm-up + 2 calls): the device IC
    generator and its VJP (2LPT), the run with three observed snapshots and the Omega_m gradient, one Adam iteration."""
    cfg, s0, p0, target = make_inputs(1, p_over_s)
    npart = s0.shape[0]
    pm = binding.PM(cfg["mesh"], cfg["lattice"], cfg["omega_m"], cfg["a"])
    omega = torch.randn(cfg["lattice"], device="cuda", generator=torch.Generator(device="cuda").manual_seed(1))
    xi, pi = torch.randn(npart, 3, device="cuda"), torch.randn(npart, 3, device="cuda")
    amp = 0.05
    rec = {"workload": cfg["name"]}
    pm.ic_fwd(omega, amp)
    rec["ic_fwd_2lpt_ms"] = _events_ms(torch, lambda: pm.ic_fwd(omega, amp), 2)
    pm.ic_vjp(omega, amp, xi, pi)
    rec["ic_vjp_2lpt_ms"] = _events_ms(torch, lambda: pm.ic_vjp(omega, amp, xi, pi), 2)
    dv = [torch.from_numpy(v).cuda() for v in (s0, p0)]
    n = cfg["n_steps"]
    tg = torch.from_numpy(np.stack([target] * 3)).cuda()
    steps, w = [n // 3, 2 * n // 3, n], [1.0, 1.0, 1.0]
    pm.run_fwd_adj_obs(dv[0], dv[1], steps, w, tg)
    rec["run_3_snapshots_ms"] = _events_ms(torch, lambda: pm.run_fwd_adj_obs(dv[0], dv[1], steps, w, tg), 2)
    rec["run_3_snapshots_dJ_dOm_ms"] = _events_ms(torch, lambda: pm.run_fwd_adj_obs(dv[0], dv[1], steps, w, tg, want_dJ_dOm=True), 2)
    pm.optimize_ic(omega, tg[0], amp, 1)
    hist = []
    rec["adam_iteration_ms"] = _events_ms(torch, lambda: hist.extend(pm.optimize_ic(omega, tg[0], amp, 2)), 1) / 2
    rec["adam_J"] = hist
    pm.close()
    return rec


def scale_up_cfg3(args, torch, binding, p_over_s, peak, peak_src, local):
    """configs[3]: 1 warm-up + 2 timed runs, an instrumented run for the kernel table, and the peak
    memory for n = 25, 50, 100 steps (north_star: peak HBM must not grow with the step count)."""
    cfg, s0, p0, target = make_inputs(3, p_over_s)
    npart = s0.shape[0]
    s0d, p0d, tgd = (torch.from_numpy(v).cuda() for v in (s0, p0, target))
    del s0, p0, target
    outs = {k: torch.empty((npart, 3), dtype=torch.float32, device="cuda") for k in ("s_n", "p_n", "xi0", "pi0", "dJ_ds0")}
    stream = torch.cuda.current_stream()
    rec = {"workload": cfg["name"], "particles": int(npart), "mesh": list(cfg["mesh"])}
    mem = {}
    for n in (25, 50, 100):
        a = inputs.a_schedule(cfg["a0"], n)
        torch.cuda.synchronize()
        torch.cuda.empty_cache()
        torch.cuda.reset_peak_memory_stats()
        free0 = torch.cuda.mem_get_info(local)[0]
        alloc0 = torch.cuda.memory_allocated()
        pm = binding.PM(cfg["mesh"], cfg["lattice"], cfg["omega_m"], a, device=f"cuda:{local}")
        smp = FreeMemSampler(torch, local)
        J = pm.run_fwd_adj(s0d, p0d, tgd, out=outs)["J"]          # also the warm-up of the n = 100 ctx
        min_free = smp.stop()
        mem[str(n)] = {"torch_peak_GB": torch.cuda.max_memory_allocated() / 1e9,
                       "torch_peak_above_inputs_GB": (torch.cuda.max_memory_allocated() - alloc0) / 1e9,
                       "memgetinfo_delta_GB": (free0 - min_free) / 1e9, "workspace_GB": pm.workspace_nbytes / 1e9}
        if n != 100:
            pm.close()
            del pm
    rec["peak_mem_vs_steps"] = mem
    rec["peak_mem_independent_of_steps"] = len({round(v["memgetinfo_delta_GB"], 2) for v in mem.values()}) == 1 and \
        len({round(v["torch_peak_GB"], 3) for v in mem.values()}) == 1
    n = 100

    def step_dev():
        return pm.run_fwd_adj(s0d, p0d, tgd, out=outs)["J"]

    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    own0, fft0 = pm.launch_count()
    clocks = ClockSampler(local)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(2):
        J = step_dev()
    e1.record(stream)
    torch.cuda.synchronize()
    clk = clocks.stop()
    own1, fft1 = pm.launch_count()
    ms = e0.elapsed_time(e1)
    rec.update({"value": job_value(1, npart, n, 2, ms), "unit": UNIT, "ms_per_step": ms / 2, "steps": 2, "warmup": 1, "kdk_steps": n,
                "gpu_launches": int(own1 - own0), "cufft_calls": int(fft1 - fft0), "clocks": clk, "objective_J": J})
    pm.timing_enable(True)
    pm.timing_reset()
    step_dev()
    kernels = kernel_table(pm.timing_read(), 1, peak)
    pm.timing_enable(False)
    pm.timing_reset()
    rec["kernels"] = kernels
    rec["roofline"] = graded_roofline(kernels, cfg["name"], peak, peak_src)
    pm.close()
    return rec


def sweep_cfg4(args, torch, binding, peak, peak_src, L):
    """configs[4]: CIC scatter / gather / weight-gradient gather of L^3 particles on a (2L)^3 mesh, clustered (20000
    Gaussian blobs at L = 512, 70 % of the particles) against uniform positions, in generation and in random memory
    order; GB/s = SURVEY section 8d algorithmic bytes / CUDA-event time, kernel only and with the binning pass."""
    N = 2 * L
    mesh, npart = (N, N, N), L ** 3
    pm = binding.PM(mesh, (L, L, L), 0.3, [1.0])
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
    steps, warm = max(3, min(args.steps, 5)), max(1, min(args.warmup, 3))

    def measure(x):
        res = {}
        for oname, op in ops.items():
            for _ in range(warm):
                op(x)
            torch.cuda.synchronize()
            pm.timing_enable(True)
            pm.timing_reset()
            for _ in range(steps):
                op(x)
            torch.cuda.synchronize()
            tm = pm.timing_read()
            pm.timing_enable(False)
            pm.timing_reset()
            k_ms = tm[cls_of[oname]]["ms"] / steps
            bin_ms = sum(tm[b]["ms"] for b in ("bin_count", "bin_scan", "bin_reorder")) / steps
            res[oname] = {"kernel_ms": k_ms, "binning_ms": bin_ms, "GBps": algo[oname] / (k_ms * 1e-3) / 1e9,
                          "frac_of_peak": algo[oname] / (k_ms * 1e-3) / 1e9 / peak,
                          "GBps_with_binning": algo[oname] / ((k_ms + bin_ms) * 1e-3) / 1e9,
                          "frac_of_peak_with_binning": algo[oname] / ((k_ms + bin_ms) * 1e-3) / 1e9 / peak}
        return res

    out = {}
    x = torch.from_numpy(inputs.blob_positions(npart, mesh, seed=3, n_blobs=n_blobs, order="generation")).cuda()
    out["clustered/generation"] = measure(x)
    perm = torch.randperm(npart, device="cuda", generator=torch.Generator(device="cuda").manual_seed(7))
    x = x[perm].contiguous()          # the same positions in a seeded random memory order
    del perm
    out["clustered/random"] = measure(x)
    del x
    x = torch.from_numpy(inputs.uniform_positions(npart, mesh, seed=3)).cuda()
    out["uniform/generation"] = measure(x)
    del x
    rec = {"workload": f"cfg4_kernel_sweep_{L}p_{N}m", "particles": npart, "mesh": list(mesh), "blobs": n_blobs, "steps": steps,
           "warmup": warm, "peak": peak, "peak_source": peak_src, "unit": "GB/s (SURVEY 8d algorithmic bytes / CUDA-event time)",
           "cases": out, "vs_uniform": {op: out["clustered/generation"][op]["GBps"] / out["uniform/generation"][op]["GBps"] for op in ops}}
    pm.close()
    return rec


def run_sweep_only(args):
    import torch
    from paper_2211_09815_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(0)
    peak, peak_src = measured_peak_gbs()
    rec = sweep_cfg4(args, torch, binding, peak, peak_src, args.sweep_lattice)
    line = {"metric": "CIC scatter/gather GB/s vs HBM peak (kernel sweep)", "value": rec["cases"]["clustered/generation"]["scatter1"]["GBps"],
            "unit": "GB/s", "n_gpus": 1, "steps": rec["steps"], "warmup": rec["warmup"], "higher_is_better": True, "dtype": "f32",
            "data": "synthetic", "vs_baseline": None, "config": {"workload": rec["workload"]}, "sweep": {"cfg4": rec},
            "peak_mem_GB": torch.cuda.max_memory_allocated() / 1e9}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs index (0-3; 4 = only the CIC kernel sweep)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-steps", type=int, default=1, help="forward + adjoint step pairs per sample of the reference arm")
    ap.add_argument("--ref-budget-s", type=float, default=480.0, help="reference arm: no further sample is started beyond this")
    ap.add_argument("--cpu-pairs", type=int, default=2, help="forward + adjoint step pairs in the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-kernel-timing", action="store_true", help="no per-kernel CUDA events pass (debug)")
    ap.add_argument("--no-scale-up", action="store_true", help="skip the configs[3] sub-record")
    ap.add_argument("--no-modes", action="store_true", help="skip the fp64-transform mode and the 8f-row timings")
    ap.add_argument("--no-sweep", action="store_true", help="skip the configs[4] sub-record")
    ap.add_argument("--sweep-lattice", type=int, default=512, help="particles per axis of the configs[4] kernel sweep (mesh = 2x)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.config == 4:
        run_sweep_only(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
