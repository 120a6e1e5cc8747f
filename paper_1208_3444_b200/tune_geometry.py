#!/usr/bin/env python
"""Launch-geometry sweep behind `choose_plain_geometry`, the one-directional force kernel's geometry
(csrc/colatus_api.cu; DESIGN.md 6.3 "Launch geometry"; the symmetric kernel is switched off for the sweep).

    python -m paper_1208_3444_b200.tune_geometry [--sizes 4096,8192,...] [--fit] > profiles/rNN_geometry_sweep.md

For every size it times the stateless force path (colatus_forces: staging + force kernel + partial-sum reduction)
through the C ABI for every kernel variant (targets per thread) and every admissible source split, forced with
colatus_set_option, CUDA events around a burst of back-to-back calls, and prints one markdown table per size
with the automatic choice marked.  --fit then fits the cost model

    time ~ a_IP * IP * S * (per_sm + ramp) + per_sm * c0,     per_sm = ceil(CTAs / SMs),  S = sources per split

to the measurements and prints the constants to paste into choose_geometry, plus how far the model's pick is
from the best measured geometry at every size.  Needs a B200; uses equal-mass inputs below 262144 bodies (the
cosmological configurations) and log-normal masses above.
"""
from __future__ import annotations

import argparse
import math
import sys

import numpy as np


def sweep(sizes, reps_us=20000.0):
    import torch
    from . import binding as B
    from . import inputs
    from .harness import Session
    rows = []
    for n in sizes:
        cfg, pm, _ = inputs.make_config(1 if n < 262144 else 4, n)
        with Session(1.0, n) as s:
            B.colatus_set_option("symmetric", 0)      # this tool sweeps the ONE-DIRECTIONAL kernel's geometry
            dev = s.to_device(pm)
            out = torch.empty_like(dev)

            def timed():
                geo = B.colatus_force_geometry(n)
                for _ in range(2):
                    B.colatus_forces(dev, n, cfg.eps2, out)
                est_us = max(float(n) * n / 2.5e6, 10.0)          # ~2500 Gint/s
                reps = int(max(3, min(200, reps_us / est_us)))
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record()
                for _ in range(reps):
                    B.colatus_forces(dev, n, cfg.eps2, out)
                e1.record()
                torch.cuda.synchronize()
                return e0.elapsed_time(e1) / reps * 1e3, geo

            us, geo = timed()
            auto = (geo["targets_per_thread"], geo["source_splits"], us)
            for tpt in (2, 4, 6):
                B.colatus_set_option("targets_per_thread", tpt)
                seen = set()
                for sp in list(range(1, 17)) + [18, 20, 24, 28, 32, 37, 40, 48, 56, 64]:
                    try:
                        B.colatus_set_option("source_splits", sp)
                    except B.ColatusError:
                        continue
                    geo = B.colatus_force_geometry(n)
                    key = (geo["source_splits"], geo["sources_per_split"])
                    if geo["source_splits"] != sp or key in seen:
                        continue
                    seen.add(key)
                    us, geo = timed()
                    rows.append({"n": n, "tpt": tpt, "splits": sp, "tiles": geo["target_tiles"],
                                 "src_per_split": geo["sources_per_split"], "us": us, "sm": geo["sm_count"]})
            B.colatus_set_option("targets_per_thread", 0)
            B.colatus_set_option("source_splits", 0)
        mine = [r for r in rows if r["n"] == n]
        best = min(mine, key=lambda r: r["us"])
        print(f"\n### N = {n}: automatic choice {auto[0]} targets/thread x {auto[1]} splits = {auto[2]:.1f} us; "
              f"best measured {best['tpt']} x {best['splits']} = {best['us']:.1f} us "
              f"({100 * (auto[2] / best['us'] - 1):+.1f} %)\n")
        print("| targets/thread | splits | CTAs | sources/split | us | Gint/s |")
        print("|---|---|---|---|---|---|")
        for r in mine:
            print(f"| {r['tpt']} | {r['splits']} | {r['tiles']} x {r['splits']} | {r['src_per_split']} | {r['us']:.1f} | "
                  f"{float(n) * n / r['us'] / 1e3:.0f} |")
        sys.stdout.flush()
    return rows


def model(p, r):
    a = {1: p[0], 2: p[1], 3: p[2]}
    ip = r["tpt"] // 2
    per_sm = math.ceil(r["tiles"] * r["splits"] / r["sm"])
    return a[ip] * ip * r["src_per_split"] * (per_sm + p[4]) + per_sm * p[3]


def fit(rows):
    from scipy.optimize import least_squares
    sol = least_squares(lambda p: [math.log(model(p, r) / r["us"]) for r in rows], [0.0274, 0.0287, 0.0295, 0.77, 0.1])
    p = sol.x
    err = np.array([math.log(model(p, r) / r["us"]) for r in rows])
    print(f"\n### Cost-model fit over {len(rows)} points\n")
    print(f"a_us[1..3] = {p[0]:.4f}, {p[1]:.4f}, {p[2]:.4f};  c0_us = {p[3]:.3f};  ramp = {p[4]:.3f};  "
          f"rms log error {err.std():.3f}, max {np.abs(err).max():.3f}\n")
    print("| N | best measured (us) | model's pick (us) | loss |")
    print("|---|---|---|---|")
    for n in sorted({r["n"] for r in rows}):
        mine = [r for r in rows if r["n"] == n]
        best = min(mine, key=lambda r: r["us"])
        pick = min(mine, key=lambda r: model(p, r))
        print(f"| {n} | {best['tpt']} x {best['splits']}: {best['us']:.1f} | {pick['tpt']} x {pick['splits']}: {pick['us']:.1f} | "
              f"{100 * (pick['us'] / best['us'] - 1):+.1f} % |")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--sizes", default="4096,8192,16384,32768,65536,131072,262144")
    ap.add_argument("--fit", action="store_true")
    args = ap.parse_args()
    sizes = [int(x) for x in args.sizes.split(",")]
    print("# Launch-geometry sweep of the force path (paper_1208_3444_b200/tune_geometry.py)\n")
    print("Command: `python -m paper_1208_3444_b200.tune_geometry --sizes " + args.sizes + (" --fit`" if args.fit else "`"))
    rows = sweep(sizes)
    if args.fit:
        fit(rows)


if __name__ == "__main__":
    main()
