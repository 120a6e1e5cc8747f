#!/usr/bin/env python
"""bench.py -- Ginteractions/s of the COLATUS hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl native|reference]

Workload (config.workload): BASELINE.json configs[3] -- N = 2^20 bodies, 64 Gaussian clusters +
50 % uniform background, log-normal masses, eps = 1e-3, synthetic and seeded
(paper_1208_3444_b200/inputs.py).  One "step" is one pass of the whole hot path (SURVEY 8a rows
a1-a7): host Friedmann mid-step values (eq. 2), colatus_step = drift + source staging (eq. 3) -> force
kernel (eq. 1) -> partial reduce + kick + drift + tracer record (eqs. 4-5), then
colatus_diagnostics (momentum / kinetic energy reductions).  N^2 pair interactions per step;
20 flop per interaction (BASELINE convention).

--impl reference times the FP64 CPU oracle (oracle/) on the host cores on a bounded sample of the
same workload; it is a deliberately slow baseline, not the target.

N > 1 (torchrun, one rank per GPU): eq. (1) sharded by targets, positions all-gathered over NCCL
after each drift (the path's only exchange step); total work fixed -> "scaling": "strong".
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

WORKLOAD_CONFIG = 4                        # BASELINE.json configs[3]: N = 2^20
FLOP_PER_INTERACTION = 20.0                # BASELINE.json convention
SM_COUNT, FP32_LANES, SM_MAX_MHZ = 148, 128, 1965.0
FP32_PEAK_TFLOPS = SM_COUNT * FP32_LANES * 2 * SM_MAX_MHZ * 1e6 / 1e12     # 74.45
# dram__bytes_read.sum + dram__bytes_write.sum of one force-kernel launch at N = 2^20 from the
# `ncu --set full` capture summarised in profiles/ (None until that capture exists).
FORCE_KERNEL_DRAM_TRAFFIC_BYTES = 130877184     # profiles/r01_force_kernel_ncu_full.txt
METRIC = "Ginteractions/s softened direct-sum gravity at N=2^20; % of FP32 FMA peak"
UNIT = "Ginteractions/s"
BENCH_TAU = 1.0e-6                         # step size of the bench steps (EdS background from a = 0.02)
N_TRACERS = 64


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-step-loops", action="store_true", help="skip the configs 1-3 steps/s side measurement")
    ap.add_argument("--config", type=int, default=WORKLOAD_CONFIG, choices=[2, 3, 4, 5],
                    help="4 = N=2^20 (the reported workload, default); 5 = N=2^22 (the at-scale case of BASELINE.json); "
                         "2, 3 = the equal-mass stepping configurations (N = 32768, 131072), for profiling the equal-mass loop")
    ap.add_argument("--n", type=int, default=0, help="override N (debug only; the reported workload is 2^20)")
    return ap.parse_args()


# --------------------------------------------------------------------------------------------------
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop_evt.wait(0.05)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# --------------------------------------------------------------------------------------------------
def oracle_sample_rate(pm, cfg, seconds_target=12.0, max_targets=65536):
    """Oracle forces on a bounded seeded sample of targets; returns (Gint/s, cores, description)."""
    import oracle
    from paper_1208_3444_b200 import inputs
    n = pm.shape[0]
    probe = inputs.sample_targets(cfg, 256)
    t0 = time.perf_counter()
    oracle.forces(pm, cfg.eps2, cfg.G, probe)
    rate = 256 * n / (time.perf_counter() - t0)
    k = int(min(max_targets, max(512, seconds_target * rate / n)))
    k = max(256, (k // 256) * 256)
    tg = inputs.sample_targets(cfg, k)
    t0 = time.perf_counter()
    oracle.forces(pm, cfg.eps2, cfg.G, tg)
    dt = time.perf_counter() - t0
    return k * n / dt / 1e9, oracle.num_threads(), f"{k} seeded targets x {n} sources (config {cfg.index}), FP64, {dt:.1f} s"


def step_loop_rates(device_index):
    """Side measurement ("steps/s for configs 1-3, CUDA graph on/off"): whole leapfrog steps per
    second of the small, launch-bound configurations through colatus_run with graph replay, the same kernels
    launched one by one from the native loop, and colatus_step called per step from Python.  Device time by
    CUDA events on the resident stream (colatus_run orders its own stream inside it); two repetitions, best."""
    import torch
    from paper_1208_3444_b200 import binding as B
    from paper_1208_3444_b200 import inputs
    from paper_1208_3444_b200.harness import Session
    out = {}
    for index, steps in ((1, 400), (2, 200), (3, 40)):
        cfg, pm, vel = inputs.make_config(index)
        row = {"n": cfg.n, "steps_timed": steps}
        with Session(cfg.G, cfg.n, device=device_index) as s:
            tau = 1e-3 * cfg.tau                       # tiny steps: the state stays near the initial one
            for mode in ("graph", "launch", "python"):
                best = None
                for _ in range(3):                     # first repetition warms up / captures
                    s.upload(pm, vel, cfg.eps2)
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    torch.cuda.synchronize()
                    e0.record()
                    if mode == "python":
                        s.run(cfg.cosmo, cfg.a_start, tau, steps)
                    else:
                        B.colatus_run(cfg.cosmo, cfg.a_start, tau, steps, mode == "graph")
                    e1.record()
                    torch.cuda.synchronize()
                    ms = e0.elapsed_time(e1)
                    best = ms if best is None else min(best, ms)
                row[mode + "_steps_per_s"] = steps / (best * 1e-3)
            row["graph_Ginteractions_per_s"] = row["graph_steps_per_s"] * float(cfg.n) ** 2 / 1e9
        out[f"config{index}"] = row
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    from paper_1208_3444_b200 import inputs
    cfg, pm, _ = inputs.make_config(args.config, args.n or None)
    n = pm.shape[0]
    k = 2048                                           # per-step sample: 2048 targets x N sources
    tg = inputs.sample_targets(cfg, k)
    for _ in range(args.warmup):
        oracle.forces(pm, cfg.eps2, cfg.G, tg[:256])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.forces(pm, cfg.eps2, cfg.G, tg)
    dt = time.perf_counter() - t0
    value = args.steps * k * n / dt / 1e9
    sample = f"{k} seeded targets x {n} sources per step (config {cfg.index}), FP64 oracle"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config {cfg.index}: N={n} clusters+background, eps={cfg.eps}", "n": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------
def run_native(args):
    from paper_1208_3444_b200 import build as cuda_build
    cuda_build.build()                      # no-op when libcolatus.so is up to date (atomic replace otherwise)
    import torch
    import torch.distributed as dist
    from paper_1208_3444_b200 import binding as B
    from paper_1208_3444_b200 import inputs
    from paper_1208_3444_b200.harness import Session
    from paper_1208_3444_b200.sharded import LibcolatusOps, ShardedStepper, partition

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl native needs a CUDA device (libcolatus has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    cfg, pm, vel = inputs.make_config(args.config, args.n or None)
    n = pm.shape[0]
    cosmo = inputs.Cosmology(H0=float(np.sqrt(8.0 * np.pi / 3.0)), Om_M=1.0)     # EdS, as config 1
    sess = Session(cfg.G, n, device=local_rank)
    begin, count = partition(n, world, rank)
    sess.upload(pm, vel, cfg.eps2)
    if world > 1:
        sess.acc = torch.zeros((count, 4), dtype=torch.float32, device=sess.device)
        ops = LibcolatusOps(sess.pos, sess.vel, sess.acc, n, cfg.eps2, begin, count)
        stepper = ShardedStepper(sess.pos, n, ops)
    tr_idx = (np.arange(N_TRACERS, dtype=np.int64) * (n // N_TRACERS)).astype(np.int32)
    sess.trace(tr_idx, max(args.steps + args.warmup, 1))
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=sess.device)       # > 126 MB L2

    state = {"a": 0.02}
    # measured denominator (register-only FMA loops through the C ABI), beside the derived 74.45 TFLOP/s
    cal_ffma, _ = B.colatus_calibrate_fp32(0)
    cal_ffma2, _ = B.colatus_calibrate_fp32(1)

    def one_step():
        a_mid = B.colatus_a_advance(cosmo, state["a"], 0.5 * BENCH_TAU)              # a1 (host, double)
        H_mid = B.colatus_hubble(cosmo, a_mid)
        if world > 1:
            stepper.step(BENCH_TAU, a_mid, H_mid)                                    # a2-a6, sharded
        else:
            B.colatus_step(BENCH_TAU, a_mid, H_mid)                                  # a2-a6
        d = B.colatus_diagnostics(a_mid, False)                                      # a7 (syncs)
        state["a"] = B.colatus_a_advance(cosmo, a_mid, 0.5 * BENCH_TAU)
        flush_buf.zero_()                                                            # L2 flush between steps
        return d

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        one_step()
    barrier()
    B.colatus_profile(True)
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = B.colatus_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        diag = one_step()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop()
    launches = B.colatus_launch_count() - launches0
    kernel_ms, kernel_launches = B.colatus_profile_read()
    B.colatus_profile(False)
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device=sess.device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_step = ms_total / args.steps
    value = float(n) * n / (ms_step * 1e-3) / 1e9

    # ---- roofline of the dominant kernel (force kernel), from events inside the timed region
    pairs_per_launch = float(count) * n
    geo = B.colatus_force_geometry(n, count)
    k_ms = kernel_ms / max(kernel_launches, 1)
    achieved = FLOP_PER_INTERACTION * pairs_per_launch / (k_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "achieved": achieved, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                "frac": achieved / FP32_PEAK_TFLOPS, "traffic": FORCE_KERNEL_DRAM_TRAFFIC_BYTES if (n == 1 << 20 and world == 1) else None,
                "kernel": "force_kernel<%d,%d,4,false,2>" % (geo["targets_per_thread"] // 2,
                                                             {6: 512, 4: 512, 2: 256}[geo["targets_per_thread"]]),
                "kernel_ms": k_ms,
                "kernel_share_of_step": k_ms / ms_step,
                "peak_basis": "derived: 148 SM x 128 FP32 lanes x 2 flop x 1965 MHz (DESIGN.md); "
                              "no FP32 figure in MEASURED_PEAKS.json",
                "peak_measured": {"ffma_tflops": cal_ffma, "ffma2_tflops": cal_ffma2,
                                  "how": "colatus_calibrate_fp32: register-only FFMA / FFMA2 loops, best of 3"},
                "frac_of_measured_peak": achieved / max(cal_ffma, cal_ffma2),
                "flop_per_interaction": FLOP_PER_INTERACTION,
                "frac_at_sampled_clock": (achieved / (FP32_PEAK_TFLOPS * clocks["sm_mhz"] / SM_MAX_MHZ)
                                          if clocks.get("sm_mhz") else None)}

    # ---- end to end through the C ABI with HOST buffers (N = 1 only: the call is single-GPU)
    e2e = None
    if world == 1:
        h_in = torch.from_numpy(pm).pin_memory()
        h_out = torch.empty((n, 4), dtype=torch.float32).pin_memory()
        B.colatus_forces_host(h_in, n, cfg.eps2, h_out)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            B.colatus_forces_host(h_in, n, cfg.eps2, h_out)          # H2D + eq. (1) + D2H + sync
        dt = time.perf_counter() - t0
        e2e = {"value": args.steps * float(n) * n / dt / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": 16 * n, "d2h_bytes_per_step": 16 * n,
               "call": "colatus_forces_host (pinned host buffers)", "ms_per_step": dt / args.steps * 1e3}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, cores, sample = oracle_sample_rate(pm, cfg)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}

    sess.close()
    step_loops = None
    if rank == 0 and world == 1 and not args.no_step_loops and not args.n and args.config == WORKLOAD_CONFIG:
        step_loops = step_loop_rates(local_rank)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"config {cfg.index} ({cfg.name}): N={n}, " +
                                   ({4: "64 Gaussian clusters + 50% uniform background, log-normal masses",
                                     5: "256 Gaussian clusters + 50% uniform background, log-normal masses",
                                     3: "Plummer sphere + 30% uniform background, equal masses",
                                     2: "32^3 lattice + Gaussian displacements, equal masses"}[cfg.index]) +
                                   f", eps={cfg.eps}; one full leapfrog step + diagnostics per step",
                       "n": n, "interactions_per_step": float(n) * n, "tracers": N_TRACERS,
                       "parallelism": "single GPU" if world == 1 else f"targets sharded over {world} GPUs, "
                                                                       "all-gather of positions per drift",
                       "l2_flush": "256 MiB memset between steps (inside the timed region)",
                       "geometry": geo},
            "gflops": value * FLOP_PER_INTERACTION,
            "frac_fp32_peak": value * FLOP_PER_INTERACTION / 1e3 / (FP32_PEAK_TFLOPS * world),
            "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e,
            "gpu_launches": int(launches), "clocks": clocks,
            "step_loops": step_loops,
            "diagnostics_last_step": {"M": diag[0], "T": diag[7]},
            "paper_context": "paper reports no timing; largest run 32^3 particles on a GTX680 (PAPER.md:23)",
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_native(a)
