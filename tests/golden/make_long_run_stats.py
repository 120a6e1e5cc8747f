#!/usr/bin/env python
"""Writes tests/golden/long_run_stats.json: the FP64 oracle's statistics of the two long runs of
BASELINE.json at their own size (reading G20, "longer runs are compared only statistically").

    python tests/golden/make_long_run_stats.py [--out tests/golden/long_run_stats.json]
                                               [--side 32] [--n3 131072] [--only 2|3]

Imports `oracle` and the seeded input generators (`paper_1208_3444_b200.inputs`) ONLY: no CUDA, no
binding, nothing of the product path.  Every number in the JSON is the oracle's.

* config 2 (PAPER.md:85-87 shape; BASELINE.json configs[1]): 32^3 lattice + Gaussian displacements, flat
  LCDM 0.3/0.7, H0 = 70, a: 1/51 -> 1 in 1000 uniform steps (readings G12, G13), 64 tracers 512*t (G18);
* config 3 (BASELINE.json configs[2]): 131072 bodies, Plummer sphere + 30 % background, static
  background, 100 steps of tau = 1e-3 (reading G13).

Each is run TWICE: run "A" from the inputs of record and run "B" from the same inputs with every position
coordinate moved by one FP32 ulp up or down (seeded).  |A - B| is the oracle's own sensitivity to an
input change below FP32 resolution: no FP32 implementation can be asked to track A more closely than B
does, so the GPU tests derive their chaotic-phase thresholds from it (tests/test_gpu_long_run.py) instead
of from a hand-picked number.

Cost: about 1.07e12 (config 2) and 1.72e12 (config 3) pair evaluations per run; minutes on 16 cores.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1208_3444_b200 import inputs  # noqa: E402

QUANTILES = [1, 5, 10, 20, 25, 30, 40, 50, 60, 70, 75, 80, 90, 95, 99]     # of the all-particle speed distribution
PERTURB_SEED = 20120817                                                       # run B
CHECKPOINTS_2 = [10, 30, 50] + list(range(100, 1001, 100))
CHECKPOINTS_3 = list(range(10, 101, 10))


# ---- statistics (definitions shared with the tests, which import this module) -------------------------------
def half_mass_radius(x, m):
    """Radius about the centre of mass that holds half the mass (equal masses: the median distance)."""
    c = (m[:, None] * x).sum(0) / m.sum()
    r = np.linalg.norm(x - c, axis=1)
    order = np.argsort(r)
    cum = np.cumsum(m[order])
    return float(r[order][np.searchsorted(cum, 0.5 * cum[-1])])


def speed_quantiles(v):
    return [float(q) for q in np.percentile(np.linalg.norm(v, axis=1), QUANTILES)]


def one_ulp_perturbed(pos_mass, seed=PERTURB_SEED):
    """Every position coordinate moved to the next FP32 value up or down (seeded coin); masses untouched."""
    rng = np.random.Generator(np.random.PCG64(seed))
    out = pos_mass.copy()
    toward = np.where(rng.random((pos_mass.shape[0], 3)) < 0.5, -np.inf, np.inf).astype(np.float32)
    out[:, :3] = np.nextafter(pos_mass[:, :3], toward)
    return out


def checkpoint_record(step, a, st, m, tr_idx=None):
    d = st.diagnostics(a, with_potential=True)
    rec = {"step": int(step), "a": float(a), "M": float(d[0]), "P": [float(d[1]), float(d[2]), float(d[3])],
           "T": float(d[7]), "W": float(d[8]), "r_half": half_mass_radius(st.x, m),
           "speed_q": speed_quantiles(st.v)}
    if tr_idx is not None:
        rec["tracer_speed"] = [float(s) for s in np.linalg.norm(st.v[tr_idx], axis=1)]
    return rec


# ---- the runs ---------------------------------------------------------------------------------------------
def config2_setup(side):
    cfg, pm, vel = inputs.make_config(2, side ** 3)
    eps2 = np.float32(np.float32(0.05 / side) ** 2)           # eps = 0.05 cell spacings (BASELINE.json configs[1])
    k = 64
    tr_idx = (np.arange(k, dtype=np.int64) * (cfg.n // k)).astype(np.int32)     # 512*t at 32^3 (G18)
    return cfg, pm, vel, eps2, tr_idx


def run_config2(side, steps, checkpoints, perturbed, log=None):
    cfg, pm, vel, eps2, tr_idx = config2_setup(side)
    if perturbed:
        pm = one_ulp_perturbed(pm)
    m = pm[:, 3].astype(np.float64)
    st = oracle.State(pm, vel, eps2, cfg.G)
    mids, ends = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, steps)
    rows = np.zeros((steps, tr_idx.size, 4), dtype=np.float32)
    recs, t0 = [], time.time()
    for n, (am, Hm) in enumerate(mids):
        st.step(cfg.tau, am, Hm)
        rows[n, :, :3] = st.v[tr_idx]                          # the ring row of step n (G18), rounded to FP32
        rows[n, :, 3] = am
        if (n + 1) in checkpoints:
            recs.append(checkpoint_record(n + 1, ends[n + 1], st, m, tr_idx))
            if log:
                log(f"config 2 {'B' if perturbed else 'A'} step {n + 1}: T={recs[-1]['T']:.6g} "
                    f"W={recs[-1]['W']:.6g} r_half={recs[-1]['r_half']:.5f} ({time.time() - t0:.0f} s)")
    spec = oracle.trace_spectrum(rows)
    return {"n": int(cfg.n), "steps": int(steps), "eps2": float(eps2), "G": float(cfg.G), "tau": float(cfg.tau),
            "a_start": float(cfg.a_start), "a_end": float(ends[-1]), "checkpoints": recs,
            "tracer_index": [int(i) for i in tr_idx],
            "tracer_rows_first10": rows[:10, :, :3].astype(np.float64).round(12).tolist(),
            "tracer_sum_v2": float((rows[:, :, :3].astype(np.float64) ** 2).sum()),
            "spectrum_power_per_tracer": [float(s) for s in spec.sum(axis=1)],
            "spectrum_power_total": float(spec.sum())}


def run_config3(n, steps, checkpoints, perturbed, log=None):
    cfg, pm, vel = inputs.make_config(3, n)
    if perturbed:
        pm = one_ulp_perturbed(pm)
    m = pm[:, 3].astype(np.float64)
    st = oracle.State(pm, vel, cfg.eps2, cfg.G)
    recs, t0 = [checkpoint_record(0, 1.0, st, m)], time.time()
    for s in range(steps):
        st.step(cfg.tau, 1.0, 0.0)                             # static background (G13)
        if (s + 1) in checkpoints:
            recs.append(checkpoint_record(s + 1, 1.0, st, m))
            if log:
                log(f"config 3 {'B' if perturbed else 'A'} step {s + 1}: T={recs[-1]['T']:.6g} "
                    f"W={recs[-1]['W']:.6g} ({time.time() - t0:.0f} s)")
    return {"n": int(cfg.n), "steps": int(steps), "eps2": float(cfg.eps2), "G": float(cfg.G), "tau": float(cfg.tau),
            "checkpoints": recs}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(ROOT, "tests", "golden", "long_run_stats.json"))
    ap.add_argument("--side", type=int, default=32)
    ap.add_argument("--n3", type=int, default=131072)
    ap.add_argument("--only", type=int, default=0, choices=[0, 2, 3])
    args = ap.parse_args()

    def log(msg):
        print(msg, flush=True)

    out = {"written_by": "tests/golden/make_long_run_stats.py (FP64 oracle only)",
           "oracle_threads": oracle.num_threads(), "quantiles": QUANTILES, "perturb_seed": PERTURB_SEED}
    if os.path.exists(args.out):                               # --only keeps the other config's block
        with open(args.out) as fh:
            out.update({k: v for k, v in json.load(fh).items() if k in ("config2", "config3")})
    if args.only in (0, 2):
        out["config2"] = {run: run_config2(args.side, 1000, CHECKPOINTS_2, run == "B", log) for run in ("A", "B")}
    if args.only in (0, 3):
        out["config3"] = {run: run_config3(args.n3, 100, CHECKPOINTS_3, run == "B", log) for run in ("A", "B")}
    tmp = args.out + ".tmp"
    with open(tmp, "w") as fh:
        json.dump(out, fh, separators=(",", ":"))
        fh.write("\n")
    os.replace(tmp, args.out)
    log(f"wrote {args.out}")


if __name__ == "__main__":
    main()
