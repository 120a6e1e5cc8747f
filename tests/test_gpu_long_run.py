"""Long runs are compared statistically (north_star: "the dynamics are chaotic and longer runs are compared only
statistically"; reading G20) -- at the configurations' OWN size and step count:

* config 2 (PAPER.md:85-87 shape): 32^3 bodies, flat LCDM, z = 50 -> 0 in 1000 uniform steps, 64 tracers;
* config 3: 131072 bodies (Plummer sphere + background), static background, 100 steps.

The FP64 oracle's side is tests/golden/long_run_stats.json, written by tests/golden/make_long_run_stats.py (oracle
and input generators only; 1.1e12 + 1.7e12 pair evaluations per run, minutes of CPU).  That file holds TWO oracle
runs per configuration: "A" from the inputs of record and "B" from inputs moved by one FP32 ulp.  |A - B| is what
the dynamics make of a perturbation below FP32 resolution, so it calibrates every threshold here; none is
hand-picked after looking at a GPU result:

    sat(statistic)             = max of |A - B| / |A| over the chaotic checkpoints (config 2: step >= 200)
    tol(statistic, checkpoint) = clip(100 * |A - B| / |A|,  1e-3,  min(3 * sat, 10 %))     before chaos has saturated
                               = min(3 * sat, 10 %)                                        at the chaotic checkpoints

* 1e-3 floor: while the flow is laminar (config 2 up to the first collapse near step 50, all of config 3) A and
  B agree to 1e-5..1e-9 and the FP32 run is held to 1e-3 -- ten times tighter than G20's "within 1 %";
* factor 100: the FP32 run is perturbed by roundoff at every step, not once, so it may sit further from A than B
  does while the difference still grows;
* 3 * sat: once chaos has saturated, GPU-vs-A is a draw from the same distribution as B-vs-A, whose largest
  value over ten checkpoints is `sat` (config 2 at 32^3: T 1.9 %, W 1.1 %, r_half 2.0 %, speed quantiles 1.6 %);
  never looser than G20's 10 %.  At a chaotic checkpoint the scale is `sat`, a property of the regime -- NOT the
  pointwise |A - B| of that checkpoint, which is one draw and can be anywhere below it: the two oracle runs happen
  to cross in W at step 800 (|A - B| / |A| = 1.0e-4 between checkpoints at 1e-2), so 100 x the pointwise value
  would hold a third rounding realisation to 1.03 % there, below the 1.1 % the oracle's own runs differ by
  elsewhere (tests/test_long_run_calibration.py asserts this spread from the committed JSON).  Every kernel the
  library can take for this run -- the one-directional and the symmetric force kernel, two different summation
  orders, i.e. two rounding realisations -- is run against the same thresholds.

The 64-tracer speed percentiles of SURVEY G20 ("median and 90th percentile within 10 %") cannot be held to a
relative bar: between the two ORACLE runs they differ by up to 17 % (median) and 21 % (p90) -- 64 samples of a
chaotic flow (tests/test_long_run_calibration.py asserts these numbers from the committed JSON).  They are
tested in the units in which their scatter is known instead: the position of the tracers' median / p90 inside the
oracle's all-particle speed distribution has a binomial standard error sigma = sqrt(q (1 - q) / 64) = 6.25 / 3.75
percentile points PER RUN; the GPU run and run A are two such draws, so their difference scatters with
sqrt(2) sigma, and the GPU run must sit within 4 sqrt(2) sigma (35 / 21 points) of where run A's tracers sit
(A and B differ by up to 10 points, 1.9 sqrt(2) sigma).  While the flow is laminar (step <= 50) every tracer's
speed is compared one by one.
"""
import importlib.util
import json
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_1208_3444_b200 import inputs  # noqa: E402
from conftest import record_parity  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
_spec = importlib.util.spec_from_file_location("make_long_run_stats",
                                               os.path.join(HERE, "golden", "make_long_run_stats.py"))
G = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(G)                      # statistic definitions shared with the script that wrote the JSON
with open(os.path.join(HERE, "golden", "long_run_stats.json")) as _fh:
    GOLD = json.load(_fh)
Q50, Q90 = G.QUANTILES.index(50), G.QUANTILES.index(90)
FLOOR, FACTOR, CAP = 1e-3, 100.0, 0.10


def _stats(rec):
    return {"T": rec["T"], "W": rec["W"], "r_half": rec["r_half"], "q50": rec["speed_q"][Q50],
            "q90": rec["speed_q"][Q90]}


def _rel(a, b):
    return abs(a - b) / max(abs(a), 1e-300)


def calibrated_tolerances(block, chaotic_from):
    """tol[statistic][checkpoint index] from the two oracle runs of `block` (see the module docstring)."""
    A, B = block["A"]["checkpoints"], block["B"]["checkpoints"]
    self_diff = {k: [_rel(_stats(a)[k], _stats(b)[k]) for a, b in zip(A, B)] for k in _stats(A[-1])}
    tol = {}
    for k, sd in self_diff.items():
        chaotic = [d for a, d in zip(A, sd) if chaotic_from is not None and a["step"] >= chaotic_from]
        cap = min(3.0 * max(chaotic), CAP) if chaotic else CAP
        tol[k] = [max(cap, FLOOR) if (chaotic_from is not None and a["step"] >= chaotic_from)
                  else min(max(FACTOR * d, FLOOR), max(cap, FLOOR)) for a, d in zip(A, sd)]
    return tol, self_diff


def _parent_percentile(value, rec):
    """Where `value` sits in the oracle's all-particle speed distribution of checkpoint `rec` (percent)."""
    return float(np.interp(value, rec["speed_q"], G.QUANTILES))


@pytest.mark.parametrize("kernel", ["symmetric", "one-directional"])
def test_config2_full_size_1000_steps_statistics(kernel):
    from paper_1208_3444_b200 import binding as B
    from paper_1208_3444_b200.harness import Session
    gold = GOLD["config2"]
    A = gold["A"]
    cfg, pm, vel, eps2, tr_idx = G.config2_setup(32)
    assert cfg.n == A["n"] == 32768 and A["steps"] == 1000 and float(eps2) == A["eps2"]
    m = pm[:, 3].astype(np.float64)
    tol, _ = calibrated_tolerances(gold, chaotic_from=200)
    checkpoints = [r["step"] for r in A["checkpoints"]]

    gpu = []
    with Session(cfg.G, cfg.n) as s:
        B.colatus_set_option("symmetric", 1 if kernel == "symmetric" else 0)     # automatic choice / never
        assert B.colatus_force_plan(cfg.n)["symmetric"] == (1 if kernel == "symmetric" else 0)
        s.upload(pm, vel, eps2)
        s.trace(tr_idx, 1000)
        a, done = cfg.a_start, 0
        for cp in checkpoints:
            a = s.run_native(cfg.cosmo, a, cfg.tau, cp - done)
            done = cp
            d = s.diagnostics(a, with_potential=True)
            pos, v = s.download()
            v3 = v[:, :3].astype(np.float64)
            gpu.append({"a": a, "T": d[7], "W": d[8], "r_half": G.half_mass_radius(pos[:, :3].astype(np.float64), m),
                        "speed_q": G.speed_quantiles(v3), "tracer_speed": np.linalg.norm(v3[tr_idx], axis=1)})
        spec_gpu = s.trace_spectrum(0, 1000)
        rows_gpu = s.trace_read(0, 1000)
    assert a == pytest.approx(1.0, abs=2e-6)                          # z = 0 reached (tau of G13)

    worst = {}
    for i, (g, r) in enumerate(zip(gpu, A["checkpoints"])):
        assert g["a"] == pytest.approx(r["a"], rel=1e-8)
        gs, rs = _stats(g), _stats(r)
        for k in gs:
            rel = _rel(rs[k], gs[k])
            phase = "laminar" if r["step"] <= 50 else "chaotic"
            worst[f"{phase}_{k}"] = max(worst.get(f"{phase}_{k}", 0.0), rel)
            assert rel <= tol[k][i], (r["step"], k, gs[k], rs[k], rel, tol[k][i])
        ts_ref = np.array(r["tracer_speed"])
        if r["step"] <= 50:                                            # laminar: tracer by tracer
            assert np.abs(g["tracer_speed"] - ts_ref).max() <= 1e-3 * np.sqrt((ts_ref ** 2).mean()), r["step"]
        else:                                                          # chaotic: two 64-sample draws, 4 sqrt(2) sigma
            for q, sigma_pts in ((50, 6.25), (90, 3.75)):
                at_gpu = _parent_percentile(np.percentile(g["tracer_speed"], q), r)
                at_ref = _parent_percentile(np.percentile(ts_ref, q), r)
                worst[f"tracer_q{q}_points"] = max(worst.get(f"tracer_q{q}_points", 0.0), abs(at_gpu - at_ref))
                assert abs(at_gpu - at_ref) <= 4.0 * np.sqrt(2.0) * sigma_pts, (r["step"], q, at_gpu, at_ref)
    record_parity(f"1000-step config 2 at 32^3 vs golden oracle run ({kernel} kernel)", **worst)

    # the run is not trivial: the box collapses onto its centre (G7) and the kinetic energy grows several-fold
    assert min(g["r_half"] for g in gpu) < 0.1 * gpu[0]["r_half"] and max(g["T"] for g in gpu) > 3 * gpu[0]["T"]

    # tracer spectra: the GPU periodogram of the GPU record equals the oracle's periodogram of the same record;
    # total power (Parseval: the sum of |v|^2 over the record) against run A within 4 sigma, sigma from the
    # per-tracer A - B differences added in quadrature
    assert np.abs(spec_gpu - oracle.trace_spectrum(rows_gpu)).max() <= 1e-10 * spec_gpu.max()
    pa, pb = np.array(A["spectrum_power_per_tracer"]), np.array(gold["B"]["spectrum_power_per_tracer"])
    sigma = float(np.sqrt(((pa - pb) ** 2).sum()))
    assert abs(spec_gpu.sum() - pa.sum()) <= 4.0 * sigma, (spec_gpu.sum(), pa.sum(), sigma)
    # the first 10 recorded steps still agree sample by sample
    rows_ref = np.array(A["tracer_rows_first10"])
    vr = np.sqrt((rows_ref ** 2).sum(2).mean())
    assert np.abs(rows_gpu[:10, :, :3] - rows_ref).max() <= 2e-4 * vr


def test_config3_full_size_100_steps_energy_and_statistics():
    """Config 3's own long run (readings G13/G20): 131072 bodies, cold start, static background, 100 steps of
    tau = 1e-3 through maximum compression (near step 50) to a virialised state.  A and B agree to 1.2e-4
    throughout (the flow stays laminar over 100 steps), so every statistic is held to 1e-3..1e-2 of run A; in the
    static limit T + W is conserved by the flow, so the GPU run is also held to an absolute energy budget."""
    from paper_1208_3444_b200.harness import Session
    gold = GOLD["config3"]
    A = gold["A"]["checkpoints"]
    cfg, pm, vel = inputs.make_config(3)
    assert cfg.n == gold["A"]["n"] == 131072 and gold["A"]["steps"] == 100
    m = pm[:, 3].astype(np.float64)
    tol, self_diff = calibrated_tolerances(gold, chaotic_from=None)
    assert max(max(v) for v in self_diff.values()) < 2e-4              # laminar: the floor / 1 % cap decide

    gpu, done = [], 0
    with Session(cfg.G, cfg.n) as s:
        s.upload(pm, vel, cfg.eps2)
        for r in A:
            if r["step"] > done:
                s.run_native(None, 1.0, cfg.tau, r["step"] - done)
                done = r["step"]
            d = s.diagnostics(1.0, with_potential=True)
            pos, v = s.download()
            gpu.append({"T": d[7], "W": d[8], "r_half": G.half_mass_radius(pos[:, :3].astype(np.float64), m),
                        "speed_q": G.speed_quantiles(v[:, :3].astype(np.float64))})
            assert np.abs(d[1:4]).max() <= 1e-5 * np.sqrt(2 * d[7] * d[0] + 1e-30) + 1e-9     # sum m v stays ~0
    assert gpu[0]["T"] == 0.0 and gpu[0]["W"] == pytest.approx(A[0]["W"], rel=1e-6)
    worst = {}
    for i, (g, r) in enumerate(zip(gpu, A)):
        if r["step"] == 0:
            continue
        gs, rs = _stats(g), _stats(r)
        for k in gs:
            scale = abs(rs["W"]) if k == "T" else abs(rs[k])           # T starts at 0: measure it against |W|
            rel = abs(gs[k] - rs[k]) / scale
            worst[k] = max(worst.get(k, 0.0), rel)
            assert rel <= min(tol[k][i], 1e-2), (r["step"], k, gs[k], rs[k], rel)
    E0 = A[0]["T"] + A[0]["W"]
    drift_gpu = max(abs(g["T"] + g["W"] - E0) / abs(E0) for g in gpu)
    drift_ref = max(abs(r["T"] + r["W"] - E0) / abs(E0) for r in A)
    record_parity("100-step config 3 at N=131072 vs golden oracle run", energy_drift_gpu=drift_gpu,
                  energy_drift_oracle=drift_ref, **{"worst_rel_" + k: v for k, v in worst.items()})
    assert drift_gpu <= max(2.0 * drift_ref, 0.02)
    assert max(r["T"] for r in A) > 0.5 * abs(A[0]["W"])               # it did collapse: T reaches the scale of |W0|
