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

N > 1 (one rank per GPU): bodies owned in slices, positions all-gathered over NCCL once per step after the first
drift; eq. (1) divided by block pairs (symmetric evaluation: every rank evaluates its share of the unordered pairs,
one all-reduce of the float4[n] partial forces) or, below 20480 bodies, by targets; diagnostics by one all-reduce;
total work fixed -> "scaling": "strong".  Under torchrun the ranks come from the environment; a plain `python bench.py --gpus N`
re-launches itself under torch.distributed.run with N ranks (and fails loudly if fewer GPUs are visible).
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
# dram__bytes_read.sum + dram__bytes_write.sum of one force-kernel launch from the `ncu --set full` capture
# summarised in profiles/: valid only for the (n, source splits) it was captured at -- reported as null otherwise.
FORCE_KERNEL_DRAM_TRAFFIC = {"bytes": 129934336, "n": 1 << 20, "splits": 8, "symmetric": 0,
                             "profile": "profiles/r02_force_kernel_ncu_full.txt"}
SYM_KERNEL_DRAM_TRAFFIC = {"bytes": 287398912 + 3657097984, "n": 1 << 20, "splits": 15, "launches": 8,
                           "profile": "profiles/r03_force_sym_kernel_cfg4_chunks.csv (sum over the 8 launches of one "
                                      "evaluation)"}
# sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active of the same captures (the hardware counter beside the
# modelled lane-op figure)
FORCE_KERNEL_FMA_PIPE_NCU = {"value": 0.883, "profile": "profiles/r02_force_kernel_ncu_full.txt"}
SYM_KERNEL_FMA_PIPE_NCU = {"value": 0.8366, "profile": "profiles/r03_force_sym_kernel_cfg4_chunk_ncu_full.txt"}
# executed floating-point operations per pair interaction (SASS count): 3 add + 3 mul + 6 fma
# (x2) + 1 rsqrt = 19 in the general loop, 18 in the equal-mass loop -- beside the 20-flop BASELINE convention
EXECUTED_FLOP_GENERAL, EXECUTED_FLOP_EQUAL_MASS = 19.0, 18.0
FMA_PIPE_LANE_OPS_GENERAL, FMA_PIPE_LANE_OPS_EQUAL_MASS = 12.0, 11.0
# symmetric kernel (each unordered pair once, applied to both bodies): per PAIR 3 add + 3 fma + rsqrt
# + 4 mul (2 for equal masses) + 6 fma = 26 (24) flop and 16 (14) FMA-pipe lane-ops, plus ~1.07 adds per pair for
# the reaction reduction (6.4 scalar adds per source and lane, 6 targets per lane); a pair is TWO interactions
def sym_work(targets_per_thread, equal_mass):
    """(executed flop, FMA-pipe lane-ops) per DELIVERED interaction of the symmetric kernel: per pair 26 (24) flop and
    16 (14) lane-ops, plus 6.4 scalar adds per (lane, source) for the reaction reduction spread over the lane's targets."""
    red = 6.4 / targets_per_thread
    return ((24.0 if equal_mass else 26.0) + red) / 2, ((14.0 if equal_mass else 16.0) + red) / 2
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
    ap.add_argument("--no-config5", action="store_true", help="skip the N = 2^22 side leg (1 warm-up + 2 timed steps)")
    ap.add_argument("--config", type=int, default=WORKLOAD_CONFIG, choices=[2, 3, 4, 5],
                    help="4 = N=2^20 (the reported workload, default); 5 = N=2^22 (the at-scale case of BASELINE.json); "
                         "2, 3 = the equal-mass stepping configurations (N = 32768, 131072), for profiling the equal-mass loop")
    ap.add_argument("--n", type=int, default=0, help="override N (debug only; the reported workload is 2^20)")
    ap.add_argument("--only-step-loop", type=int, default=0, choices=[0, 1, 2, 3],
                    help="profiling aid: run only the colatus_run step loop of this configuration (optionally with --n) "
                         "and print its steps/s as one JSON line -- the launches ncu captures for the small-N kernels")
    ap.add_argument("--symmetric-rows", type=int, default=0,
                    help="measurement aid: cap on the partial rows one launch of the symmetric kernel may use "
                         "(colatus_set_option symmetric_rows; 0 = what the workspace holds) -- the sweep behind the "
                         "default row budget, profiles/r03_workspace_rows_sweep.md")
    ap.add_argument("--sharded-driver", action="store_true",
                    help="run the multi-GPU step driver (sharded.py) even at N = 1: a self-test of that code path on one GPU")
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


def oracle_all_pairs_rates():
    """"oracle timing ... all pairs for configs 1-3" -- the oracle as it stands, every target of each
    configuration, on the host cores (about 5 s in all)."""
    import oracle
    from paper_1208_3444_b200 import inputs
    out = {}
    for index in (1, 2, 3):
        cfg, pm, _ = inputs.make_config(index)
        t0 = time.perf_counter()
        oracle.forces(pm, cfg.eps2, cfg.G)
        dt = time.perf_counter() - t0
        out[f"config{index}"] = {"n": cfg.n, "value": float(cfg.n) ** 2 / dt / 1e9, "unit": UNIT, "seconds": dt,
                                 "cores": oracle.num_threads(), "kind": "oracle",
                                 "sample": f"all {cfg.n} targets x {cfg.n} sources, FP64"}
    return out


def step_loop_rates(device_index, only=None, n_override=None):
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
        if only and index != only:
            continue
        cfg, pm, vel = inputs.make_config(index, n_override if only else None)
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
        "config": {"workload": workload_text(cfg, n), "n": n, "interactions_per_step": float(n) * n,
                   "sampled": f"each step evaluates {k} seeded targets x all {n} sources (a bounded sample of the "
                              "workload's N^2 interactions)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------
WORKLOAD_TEXT = {4: "64 Gaussian clusters + 50% uniform background, log-normal masses",
                 5: "256 Gaussian clusters + 50% uniform background, log-normal masses",
                 3: "Plummer sphere + 30% uniform background, equal masses",
                 2: "32^3 lattice + Gaussian displacements, equal masses"}


def workload_text(cfg, n):
    """config.workload: ONE string for the native and the reference arm (the driver compares them)."""
    return (f"config {cfg.index} ({cfg.name}): N={n}, " + WORKLOAD_TEXT[cfg.index] +
            f", eps={cfg.eps}; one full leapfrog step + diagnostics per step")


def relaunch_with_ranks(args):
    """`python bench.py --gpus N` without torchrun: start N ranks (one per GPU) of this same command under
    torch.distributed.run on 127.0.0.1 and replace this process with it.  Fails loudly if the box has fewer GPUs."""
    import socket
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit(f"bench.py --gpus {args.gpus}: only {have} CUDA device(s) visible; refusing to run fewer "
                         "ranks than requested (the sharded path needs one GPU per rank)")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def measure(args, config_index, n_override, steps, warmup, world, rank, local_rank, with_e2e):
    """W warm-up + K timed passes of the whole hot path on one configuration; returns the pieces of the JSON line."""
    import torch
    import torch.distributed as dist
    from paper_1208_3444_b200 import binding as B
    from paper_1208_3444_b200 import inputs
    from paper_1208_3444_b200.harness import Session
    from paper_1208_3444_b200.sharded import LibcolatusOps, ShardedStepper, partition

    cfg, pm, vel = inputs.make_config(config_index, n_override)
    n = pm.shape[0]
    cosmo = inputs.Cosmology(H0=float(np.sqrt(8.0 * np.pi / 3.0)), Om_M=1.0)     # EdS, as config 1
    sess = Session(cfg.G, n, device=local_rank)
    begin, count = partition(n, world, rank)
    if args.symmetric_rows:
        B.colatus_set_option("symmetric_rows", args.symmetric_rows)
    sess.upload(pm, vel, cfg.eps2)
    tr_idx = (np.arange(N_TRACERS, dtype=np.int64) * (n // N_TRACERS)).astype(np.int32)
    stepper = None
    if world > 1 or args.sharded_driver:
        sess.acc = torch.zeros((count, 4), dtype=torch.float32, device=sess.device)
        ops = LibcolatusOps(sess.pos, sess.vel, sess.acc, n, cfg.eps2, begin, count)
        stepper = ShardedStepper(sess.pos, n, ops)
    sess.trace(tr_idx, max(steps + warmup, 1))
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=sess.device)       # > 126 MB L2
    state = {"a": 0.02}

    def one_step():
        a_mid = B.colatus_a_advance(cosmo, state["a"], 0.5 * BENCH_TAU)              # a1 (host, double)
        H_mid = B.colatus_hubble(cosmo, a_mid)
        if stepper is not None:
            stepper.step(BENCH_TAU, a_mid, H_mid)                                    # a2-a6, sharded; 1 all-gather
            d = stepper.diagnostics(a_mid, False)                                    # a7: 1 all-reduce (syncs)
        else:
            B.colatus_step(BENCH_TAU, a_mid, H_mid)                                  # a2-a6
            d = B.colatus_diagnostics(a_mid, False)                                  # a7 (syncs)
        state["a"] = B.colatus_a_advance(cosmo, a_mid, 0.5 * BENCH_TAU)
        flush_buf.zero_()                                                            # L2 flush between steps
        return d

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        one_step()
    barrier()
    B.colatus_profile(True)
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = B.colatus_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(steps):
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
    ms_step = ms_total / steps
    value = float(n) * n / (ms_step * 1e-3) / 1e9

    # ---- roofline of the dominant kernel (force kernel), from events inside the timed region
    pairs_per_launch = float(count) * n
    sharded_sym = stepper is not None and stepper.symmetric       # N > 1: every rank evaluates its share of the pairs
    geo = B.colatus_force_geometry(n, n if sharded_sym else count)
    plan = B.colatus_force_plan(n, n if sharded_sym else count)
    geo["plan"] = plan
    sym = bool(plan["symmetric"])
    equal_mass = bool(np.all(pm[:, 3] == pm[0, 3]))
    k_ms = kernel_ms / max(kernel_launches, 1)
    per_s = pairs_per_launch / (k_ms * 1e-3)
    achieved = FLOP_PER_INTERACTION * per_s / 1e12
    algorithmic_bytes = 32 * n
    if sym:
        cap = SYM_KERNEL_DRAM_TRAFFIC
        traffic = cap["bytes"] if (cap and n == cap["n"] and world == 1 and plan["splits"] == cap["splits"] and
                                   plan["launches"] == cap.get("launches", 1)) else None
        executed, lane_ops = sym_work(geo["targets_per_thread"], equal_mass)
        # workspace traffic the method does not ask for: the staged copy, the target-side rows of the splits (once per
        # launch) and one reaction row per block distance
        workspace_bytes_written = 16 * plan["padded_bodies"] * (1 + plan["splits"] * plan["launches"] + plan["distances"])
        pipe_ncu = SYM_KERNEL_FMA_PIPE_NCU if traffic else None
        kernel = "force_sym_kernel<%d,%d,4,%d,%s> (every pair once, applied to both bodies)%s%s" % (
            geo["targets_per_thread"] // 2, 256 if geo["targets_per_thread"] == 4 else 512,
            1 if geo["targets_per_thread"] > 6 else 2,
            ("2" if equal_mass else "1") if plan["padded_bodies"] >= 98304 else "0",
            " equal-mass loop" if equal_mass else "",
            "; %d launches + partial-row reductions per evaluation" % plan["launches"] if plan["launches"] > 1 else "")
        if sharded_sym:
            kernel += "; share %d of %d of the block pairs per rank, one all-reduce of the partial forces" % (rank, world)
    else:
        cap = FORCE_KERNEL_DRAM_TRAFFIC
        traffic = cap["bytes"] if (n == cap["n"] and world == 1 and geo["source_splits"] == cap["splits"]) else None
        lane_ops = FMA_PIPE_LANE_OPS_EQUAL_MASS if equal_mass else FMA_PIPE_LANE_OPS_GENERAL
        executed = EXECUTED_FLOP_EQUAL_MASS if equal_mass else EXECUTED_FLOP_GENERAL
        workspace_bytes_written = 16 * n * (1 + (geo["source_splits"] if geo["source_splits"] > 1 else 0))
        pipe_ncu = FORCE_KERNEL_FMA_PIPE_NCU if traffic else None
        kernel = "force_kernel<%d,%d,4,false,2>%s" % (geo["targets_per_thread"] // 2,
                                                      {6: 512, 4: 512, 2: 128}[geo["targets_per_thread"]],
                                                      " equal-mass loop" if equal_mass else "")
    roofline = {"bound": "alu", "achieved": achieved, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                "frac": achieved / FP32_PEAK_TFLOPS, "traffic": traffic,
                "traffic_from": cap["profile"] if traffic else None,
                "algorithmic_bytes": algorithmic_bytes,
                "algorithmic_bytes_basis": "SURVEY 8(d): read N bodies + write N forces = 32 N bytes per evaluation",
                "workspace_bytes_written": workspace_bytes_written,
                "traffic_over_algorithmic": traffic / algorithmic_bytes if traffic else None,
                "kernel": kernel,
                "kernel_ms": k_ms,
                "kernel_share_of_step": k_ms / ms_step,
                "peak_basis": "derived: 148 SM x 128 FP32 lanes x 2 flop x 1965 MHz (DESIGN.md); "
                              "no FP32 figure in MEASURED_PEAKS.json",
                "flop_per_interaction": FLOP_PER_INTERACTION,
                "frac_note": ("achieved = ALGORITHMIC flops: 20 flop x N^2 pair interactions delivered / kernel time "
                              "(BASELINE convention)." + (" The symmetric kernel evaluates each unordered pair once "
                              "and applies it to both bodies, so it EXECUTES ~13.2 flop per delivered interaction: "
                              "frac (= algorithmic_frac) can exceed 20/24 = 0.833, the ceiling of a one-directional "
                              "kernel, and 1; the hardware utilisation figures are frac_executed_flops (SASS flop "
                              "count x rate), fma_pipe_busy_frac_modelled (lane-ops x rate) and "
                              "fma_pipe_busy_frac_ncu (sm__pipe_fma_cycles_active of the committed capture)."
                              if sym else "")),
                "frac_executed_flops": executed * per_s / 1e12 / FP32_PEAK_TFLOPS,
                "fma_pipe_busy_frac_modelled": lane_ops * per_s / (SM_COUNT * FP32_LANES * SM_MAX_MHZ * 1e6),
                "fma_pipe_busy_frac_ncu": pipe_ncu["value"] if pipe_ncu else None,
                "fma_pipe_busy_frac_ncu_from": pipe_ncu["profile"] if pipe_ncu else None,
                "algorithmic_frac": achieved / FP32_PEAK_TFLOPS,
                "frac_at_sampled_clock": (achieved / (FP32_PEAK_TFLOPS * clocks["sm_mhz"] / SM_MAX_MHZ)
                                          if clocks.get("sm_mhz") else None)}

    # ---- end to end through the C ABI with HOST buffers (N = 1 only: the call is single-GPU)
    e2e = None
    if world == 1 and with_e2e:
        h_in = torch.from_numpy(pm).pin_memory()
        h_out = torch.empty((n, 4), dtype=torch.float32).pin_memory()
        B.colatus_forces_host(h_in, n, cfg.eps2, h_out)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(steps):
            B.colatus_forces_host(h_in, n, cfg.eps2, h_out)          # H2D + eq. (1) + D2H + sync
        dt = time.perf_counter() - t0
        e2e = {"value": steps * float(n) * n / dt / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": 16 * n, "d2h_bytes_per_step": 16 * n,
               "call": "colatus_forces_host (pinned host buffers)", "ms_per_step": dt / steps * 1e3}
    sess.close()
    return {"cfg": cfg, "pm": pm, "n": n, "value": value, "ms_step": ms_step, "roofline": roofline, "e2e": e2e,
            "launches": int(launches), "clocks": clocks, "geo": geo, "diag": diag}


def run_native(args):
    world_env = os.environ.get("WORLD_SIZE")
    if args.gpus > 1 and world_env is None:
        relaunch_with_ranks(args)                # does not return
    from paper_1208_3444_b200 import build as cuda_build
    cuda_build.build()                      # no-op when the libraries are up to date (atomic replace otherwise)
    import torch
    import torch.distributed as dist
    from paper_1208_3444_b200 import probe as P

    world = int(world_env or "1")
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; launch one rank per GPU")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl native needs a CUDA device (libcolatus has no CPU fallback)")
    if torch.cuda.device_count() <= local_rank:
        raise SystemExit(f"bench.py: rank {rank} has no GPU (LOCAL_RANK={local_rank}, "
                         f"{torch.cuda.device_count()} visible)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    if args.only_step_loop:
        print(json.dumps({"step_loops": step_loop_rates(local_rank, args.only_step_loop, args.n or None)}), flush=True)
        return

    # measured denominator (register-only FMA loops of libcolatus_probe), beside the derived 74.45 TFLOP/s
    cal_ffma, _ = P.fp32_peak(False, local_rank)
    cal_ffma2, _ = P.fp32_peak(True, local_rank)

    m = measure(args, args.config, args.n or None, args.steps, args.warmup, world, rank, local_rank, True)
    cfg, pm, n = m["cfg"], m["pm"], m["n"]
    roofline = m["roofline"]
    roofline["peak_measured"] = {"ffma_tflops": cal_ffma, "ffma2_tflops": cal_ffma2,
                                 "how": "libcolatus_probe: register-only FFMA / FFMA2 loops, best of 3"}
    roofline["frac_of_measured_peak"] = roofline["achieved"] / max(cal_ffma, cal_ffma2)

    cpu_baseline = None
    cpu_baseline_configs = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, cores, sample = oracle_sample_rate(pm, cfg)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
        if not args.n and args.config == WORKLOAD_CONFIG:
            cpu_baseline_configs = oracle_all_pairs_rates()

    default_run = world == 1 and not args.n and args.config == WORKLOAD_CONFIG
    step_loops = None
    if rank == 0 and default_run and not args.no_step_loops:
        step_loops = step_loop_rates(local_rank)

    # side leg: the at-scale case of BASELINE.json (configs[4], N = 2^22): 1 warm-up + 2 timed steps
    config5 = None
    if rank == 0 and default_run and not args.no_config5:
        del pm
        m5 = measure(args, 5, None, 2, 1, 1, 0, local_rank, False)
        config5 = {"n": m5["n"], "steps": 2, "warmup": 1, "ms_per_step": m5["ms_step"], "value": m5["value"],
                   "unit": UNIT, "frac": m5["roofline"]["frac"], "kernel_ms": m5["roofline"]["kernel_ms"],
                   "kernel": m5["roofline"]["kernel"], "geometry": m5["geo"],
                   "clocks": m5["clocks"]}

    if rank == 0:
        value = m["value"]
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": m["ms_step"], "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_text(cfg, n),
                       "n": n, "interactions_per_step": float(n) * n, "tracers": N_TRACERS,
                       "parallelism": "single GPU" if world == 1 else f"eq. (1) divided over {world} GPUs (symmetric "
                                                                       "evaluation: by block pairs, one all-reduce of "
                                                                       "the partial forces per step; else by targets), "
                                                                       "one all-gather of positions per step, "
                                                                       "one all-reduce of 16 doubles for the diagnostics",
                       "l2_flush": "256 MiB memset between steps (inside the timed region)",
                       "geometry": m["geo"]},
            "gflops": value * FLOP_PER_INTERACTION,
            "frac_fp32_peak": value * FLOP_PER_INTERACTION / 1e3 / (FP32_PEAK_TFLOPS * world),
            "roofline": roofline, "cpu_baseline": cpu_baseline, "cpu_baseline_configs": cpu_baseline_configs,
            "e2e": m["e2e"],
            "gpu_launches": m["launches"], "clocks": m["clocks"],
            "step_loops": step_loops, "config5": config5,
            "diagnostics_last_step": {"M": float(m["diag"][0]), "T": float(m["diag"][7])},
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
