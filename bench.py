#!/usr/bin/env python
"""bench.py -- V-cycles/s of the B200 multigrid pressure solve on BASELINE config 3.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Workload (config.workload): BASELINE.json configs[2], the configuration the metric is quoted on:
256^3 fp32 rising-bubble volume fraction (density ratio 1000:1), RHS = FE divergence of a seeded
N(0,1) velocity field, 7-level V(2,2) cycle, omega = 2/3, 50 coarse sweeps.  Inputs are seeded
and synthetic (workloads/configs.py); they stand in for the paper's rising-bubble case.

One step = one V-cycle (rows a1-a6 of the hot path) on device-resident fields, launched through
the C ABI (mg_vcycle).  `value` = V-cycles/s over all ranks (replicas only: the path does not
shard); `e2e` = the same metric through mg_solve_host_zero with HOST buffers
(H2D of b, zero guess, 20 cycles -- the paper's fixed count, P:429 -- D2H of x inside the timed region).
`roofline` is for the dominant kernel, timed live with CUDA events by mg_vcycle_timed on the
solver's stream.  `cpu_baseline` is the fp64 oracle (oracle/oracle.c), as it stands, on the host
cores.  `--impl reference` times that oracle alone (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "multigrid V-cycles/s at 256^3 fp32 (V(2,2), 7 levels, variable coefficient 1/rho)"
UNIT = "V-cycles/s"
E2E_CYCLES = 20          # the paper's fixed cycle count per pressure solve
REF_TIME_BUDGET_S = 150  # wall-clock cap of the oracle arm
# roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum of one fine-level smoother launch, from the ncu --set full
# capture recorded in TRAFFIC_FILE together with the SHA-256 of the kernel source it was taken from; when the source has
# changed since, the number is stale and `traffic` is null (the file names the profile summary it belongs to)
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "traffic_lean_sweep.json")
KERNEL_SOURCES = [os.path.join(ROOT, "paper_2401_06755_b200", "csrc", f) for f in ("lean_kernel.cuh", "lean_body.inc")]


def kernel_source_sha256():
    import hashlib
    h = hashlib.sha256()
    for path in KERNEL_SOURCES:
        with open(path, "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def load_traffic():
    """(bytes per launch or None, note)"""
    try:
        with open(TRAFFIC_FILE) as f:
            d = json.load(f)
        sha = kernel_source_sha256()
    except (OSError, ValueError) as e:
        return None, "no traffic record (%s)" % e
    if d.get("source_sha256") != sha:
        return None, "stale: %s was captured from another version of lean_kernel.cuh / lean_body.inc" % d.get("from", TRAFFIC_FILE)
    return float(d["dram_bytes_per_launch"]), d.get("from", TRAFFIC_FILE)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def build_workload():
    from workloads import configs
    return configs.config3()


def algorithmic_bytes_per_cycle(w, info):
    """Bytes one fused V(nu1,nu2) cycle must move: per level point,
    down leg reads x, k, b and writes x plus 1/8 (b_c, x_c) = 17 B, up leg reads x, k, b, x_c/8 and
    writes x = 16.5 B (fp32, variable k); the coarsest level is on-chip apart from load/store."""
    total = 0.0
    for l, n in enumerate(info):
        total += n * (17.0 + 16.5) if l < len(info) - 1 else n * 16.0
    return total


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU during the timed region (pynvml)."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None
        self.ok = True

    def run(self):
        try:
            self._run_nvml()
        except Exception:
            try:
                self._run_smi()
            except Exception:
                self.ok = False

    def _run_nvml(self):
        import pynvml as nv
        nv.nvmlInit()
        h = nv.nvmlDeviceGetHandleByIndex(self.index)
        self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
        names = {
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        while not self.stop_flag:
            self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
            try:
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.02)

    def _run_smi(self):
        """No pynvml on this machine: poll nvidia-smi (B200_PROFILING.md's clocks line), one process per sample."""
        import subprocess
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        self.source = "nvidia-smi"
        while True:
            out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q, "--format=csv,noheader,nounits"],
                                 capture_output=True, text=True, timeout=10).stdout.strip().splitlines()
            f = [c.strip() for c in out[0].split(",")]
            self.samples.append(float(f[0]))
            self.max_mhz = float(f[1])
            for name, val in zip(names, f[2:]):
                if val.lower().startswith("active"):
                    self.reasons.add(name)
            if self.stop_flag:
                break
            time.sleep(0.02)

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples), "source": getattr(self, "source", "nvml")}


def max_over_ranks(ms, world, device=None):
    """Replicas only: the job's time is the slowest rank's, taken on the device timeline."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank, ms, world, device=None):
    """Whole-job throughput of `world` independent replicas: all ranks' units over the slowest rank's time."""
    return world * units_per_rank / (max_over_ranks(ms, world, device) * 1e-3)


def time_oracle(w, alpha32, b32, cycles, budget_s):
    """The oracle as it stands (fp64, OpenMP over z) on the host cores: `cycles` V-cycles of the workload."""
    import oracle
    oracle.build()
    g = oracle.grid(w.nx, w.ny, w.nz, w.h)
    k = oracle.k_from_vof(alpha32.astype(np.float64), w.rho_l, w.rho_g)
    b = b32.astype(np.float64)
    x = np.zeros(w.shape)
    done, t0 = 0, time.perf_counter()
    while done < cycles:
        x = oracle.vcycle(g, w.bc, k, x, b, w.levels, w.nu_pre, w.nu_post, w.coarse_sweeps, w.omega)
        done += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    return done / dt, done, oracle.num_threads()


def oracle_rhs(w):
    import oracle
    oracle.build()
    g = oracle.grid(w.nx, w.ny, w.nz, w.h)
    return oracle.pressure_rhs(g, w.fields["u"], w.fields["v"], w.fields["w"], 1.0).astype(np.float32)


def bench_config(w, args, world):
    """The `config` object of both arms (same keys and values, so that the driver can compare them)."""
    return {"workload": "config3_rising_bubble_256^3 (BASELINE.json configs[2])", "grid": [w.nx, w.ny, w.nz],
            "levels": w.levels, "cycle": "V(%d,%d)" % (w.nu_pre, w.nu_post), "omega": w.omega,
            "coarse_sweeps": w.coarse_sweeps, "bc": "Neumann x5, Dirichlet top", "sweeps_per_pass": args.sweeps_per_pass,
            "cycles_per_defect": args.cycles_per_defect,
            "l2_policy": "inputs larger than L2 (x, b, k = 192 MiB > 126 MB)", "parallelism": "replicas x%d" % world}


def run_reference(args, rank):
    if rank != 0:
        return
    w = build_workload()
    alpha32 = w.fields["alpha"].astype(np.float32)
    b32 = oracle_rhs(w)
    if args.warmup > 0:
        time_oracle(w, alpha32, b32, 1, 1.0)   # one untimed cycle: pages in the arrays and the OpenMP team
    value, done, cores = time_oracle(w, alpha32, b32, max(args.steps, 1), REF_TIME_BUDGET_S)
    sample = "%d V-cycle(s) of config 3 at full size (256^3, 7 levels, V(2,2)), fp64 oracle" % done
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "steps_timed": done, "warmup": args.warmup, "warmup_done": min(args.warmup, 1), "ms_per_step": 1e3 / value,
        "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": bench_config(w, args, args.gpus),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args, rank, local_rank, world):
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    import paper_2401_06755_b200 as mg

    w = build_workload()
    dev = torch.device("cuda", local_rank)
    alpha = torch.from_numpy(w.fields["alpha"].astype(np.float32)).to(dev)
    u, v, ww = (torch.from_numpy(w.fields[q].astype(np.float32)).to(dev) for q in ("u", "v", "w"))
    b = torch.empty_like(alpha)
    mg.pressure_rhs(u, v, ww, w.h, 1.0, b)            # RHS = FE divergence of the seeded velocity (product kernel)
    del u, v, ww
    s = mg.mg_create((w.nx, w.ny, w.nz, w.h), w.levels, w.bc, mg.MG_F32)
    mg.mg_set_params(s, nu_pre=w.nu_pre, nu_post=w.nu_post, coarse_sweeps=w.coarse_sweeps, sweeps_per_pass=args.sweeps_per_pass,
                     omega=w.omega, mixed_precision=1, cycles_per_defect=args.cycles_per_defect)
    mg.mg_set_coefficient_from_vof(s, alpha, w.rho_l, w.rho_g)
    x = torch.zeros_like(b)
    info = [mg.mg_level_info(s, l)[0] for l in range(w.levels)]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        mg.mg_vcycle(s, x, b)
    vis = os.environ.get("CUDA_VISIBLE_DEVICES", "").split(",")
    nvml_index = int(vis[local_rank]) if len(vis) > local_rank and vis[local_rank].strip().isdigit() else local_rank
    sampler = ClockSampler(nvml_index)
    barrier()
    sampler.start()
    l0 = mg.mg_launch_count(s)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        mg.mg_vcycle(s, x, b)
    e1.record()
    barrier()
    sampler.stop_flag = True
    launches = mg.mg_launch_count(s) - l0
    ms = e0.elapsed_time(e1)
    ms = max_over_ranks(ms, world, dev)
    sampler.join(timeout=2.0)
    value = world * args.steps / (ms * 1e-3)
    lups_per_cycle = sum(n * (w.nu_pre + w.nu_post) for n in info[:-1]) + info[-1] * w.coarse_sweeps
    glups = value * lups_per_cycle * 1e-9

    # per-level timing (CUDA events on the solver's stream, same K cycles) -> roofline of the dominant kernel
    roofline, per_level = None, None
    try:
        dn = np.zeros(w.levels); up = np.zeros(w.levels)
        reps = max(3, min(args.steps, 50))
        for _ in range(reps):
            a, c = mg.mg_vcycle_timed(s, x, b)
            dn += a; up += c
        dn /= reps; up /= reps
        per_level = [{"level": l, "points": info[l], "ms_down": float(dn[l]), "ms_up": float(up[l]),
                      "alg_bytes": info[l] * (33.5 if l < w.levels - 1 else 16.0)} for l in range(w.levels)]
        peak, peak_src = load_peaks()
        # dominant kernel: the fine-level smoother pass (5 of the 6 fine-level passes of a V(2,2) cycle are
        # this kernel or its PRO / RR variants).  Timed alone, back to back, with CUDA events on the solver's
        # stream: `nsw` sweeps in one mg_smooth call = nsw / sweeps_per_pass launches, ping-pong between x and
        # the solver's scratch (nsw even: no copy back).  Algorithmic bytes: x, k, b read + x written = 16 B
        # per point per pass.
        nsw = 20 * args.sweeps_per_pass
        xs = x.clone()
        mg.mg_smooth(s, xs, b, nsw)
        torch.cuda.synchronize()
        e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e2.record()
        mg.mg_smooth(s, xs, b, nsw)
        e3.record()
        torch.cuda.synchronize()
        launches_sm = nsw // args.sweeps_per_pass
        traffic, traffic_src = load_traffic()
        t_ms = e2.elapsed_time(e3) / launches_sm
        nbytes = 16.0 * info[0]
        achieved = nbytes / (t_ms * 1e-3) * 1e-9
        roofline = {"bound": "hbm", "kernel": "fine-level smoother pass (%d sweep(s) per launch)" % args.sweeps_per_pass,
                    "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                    "peak_source": peak_src, "alg_bytes_per_launch": nbytes, "ms_per_launch": float(t_ms),
                    "launches_timed": launches_sm}
        del xs
    except mg.MgError as e:   # instrumentation not available on this path: say so instead of inventing a number
        roofline = {"bound": "hbm", "achieved": None, "peak": load_peaks()[0], "unit": "GB/s", "frac": None,
                    "traffic": None, "note": str(e)}

    # end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    # (the solve starts from a zero guess, as the pressure correction of a time step does: only b travels to the device)
    hx = torch.empty(w.shape, dtype=torch.float32).pin_memory()
    hb = b.cpu().pin_memory()
    mg.mg_solve_host_zero(s, hx, hb, 0.0, 2)
    calls = max(2, min(10, args.steps // E2E_CYCLES))
    barrier()
    t0 = time.perf_counter()
    e0.record()
    for _ in range(calls):
        mg.mg_solve_host_zero(s, hx, hb, 0.0, E2E_CYCLES)
    e1.record()
    barrier()
    ms_e2e = e0.elapsed_time(e1)
    ms_e2e = max_over_ranks(ms_e2e, world, dev)
    e2e = {"value": world * calls * E2E_CYCLES / (ms_e2e * 1e-3), "unit": UNIT,
           "h2d_bytes_per_step": hb.numel() * 4, "d2h_bytes_per_step": hx.numel() * 4,
           "step": "one mg_solve_host_zero call = %d V-cycles from a zero guess, fp64 defect and residual norm every %s cycle(s)"
                   % (E2E_CYCLES, "4 (cycles_per_defect 0 = adaptive; fixed count)" if args.cycles_per_defect == 0 else str(args.cycles_per_defect)),
           "calls": calls}

    # config 5 (BASELINE.json configs[4]): full time step on 256^3 (momentum predictor x2, pressure RHS, mixed-precision
    # multigrid solve to 1e-6, projection, VoF update) through flow_time_step -- reported as an extra, not the headline
    time_step = None
    if rank == 0 and world == 1 and not args.no_extras:
        from workloads import configs
        w5 = configs.config5()
        f32 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
        C5, u5, v5, w5w = (f32(w5.fields[q]) for q in ("alpha", "u", "v", "w"))
        p5 = torch.empty_like(C5)
        mg.mg_set_params(s, nu_pre=w5.nu_pre, nu_post=w5.nu_post, coarse_sweeps=w5.coarse_sweeps, sweeps_per_pass=1,
                         omega=w5.omega, mixed_precision=1, cycles_per_defect=args.cycles_per_defect)
        cyc5 = []
        for it in range(2 + 5):
            if it == 2:
                torch.cuda.synchronize(); e0.record()
            st5, c5, r5 = mg.flow_time_step(s, C5, u5, v5, w5w, p5, w5.rho_l, w5.rho_g, w5.mu_l, w5.mu_g, w5.dt, w5.tol, 100)
            cyc5.append(c5)
        e1.record(); torch.cuda.synchronize()
        ms5 = e0.elapsed_time(e1) / 5
        time_step = {"workload": "config5_time_step_256^3 (BASELINE.json configs[4])", "value": 1e3 / ms5, "unit": "time-steps/s",
                     "ms_per_step": ms5, "steps_timed": 5, "warmup": 2, "cycles_per_solve": cyc5[2:], "last_status": int(st5),
                     "cycles_per_defect": args.cycles_per_defect,
                     "last_relres": float(r5), "tol": w5.tol}
        # the same steps with the pressure solved by V-cycle-preconditioned CG (flow_time_step_pcg; not in the paper)
        C5, u5, v5, w5w = (f32(w5.fields[q]) for q in ("alpha", "u", "v", "w"))
        it5 = []
        for it in range(2 + 5):
            if it == 2:
                torch.cuda.synchronize(); e0.record()
            st5, c5, r5 = mg.flow_time_step_pcg(s, C5, u5, v5, w5w, p5, w5.rho_l, w5.rho_g, w5.mu_l, w5.mu_g, w5.dt, w5.tol, 100)
            it5.append(c5)
        e1.record(); torch.cuda.synchronize()
        ms5 = e0.elapsed_time(e1) / 5
        time_step["pcg"] = {"value": 1e3 / ms5, "unit": "time-steps/s", "ms_per_step": ms5, "iterations_per_solve": it5[2:],
                            "last_status": int(st5), "last_relres": float(r5)}
        del C5, u5, v5, w5w, p5

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        val, done, cores = time_oracle(w, w.fields["alpha"].astype(np.float32), hb.numpy(), 2, 60.0)
        cpu = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "%d V-cycle(s) of the same 256^3 workload, fp64 oracle with OpenMP" % done}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": bench_config(w, args, args.gpus),
            "glups": glups, "lups_per_cycle": lups_per_cycle,
            "alg_bytes_per_cycle": algorithmic_bytes_per_cycle(w, info),
            "effective_gbs": algorithmic_bytes_per_cycle(w, info) * (args.steps / (ms * 1e-3)) * 1e-9,
            "clocks": sampler.summary(), "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "per_level": per_level, "time_step": time_step, "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    mg.mg_destroy(s)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the config-5 time-step measurement")
    ap.add_argument("--sweeps-per-pass", type=int, default=1, choices=[1, 2, 3, 4],
                    help="stencil stages per launch on a level: 1 = one-stage streaming kernels (default, faster); "
                         "2-4 = wave kernel (temporal blocking through L2)")
    ap.add_argument("--cycles-per-defect", type=int, default=0,
                    help="mixed-precision solves (e2e, time step): V-cycles per fp64 defect / residual check (mg_params.cycles_per_defect); "
                         "0 (default) = adaptive: chosen by the solve loop from the contraction it observes, 4 for a fixed cycle count")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.warmup < 3:
        args.warmup = 3
    run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
