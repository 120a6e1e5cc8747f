"""CPU side of the long-run comparison (reading G20): where the thresholds of tests/test_gpu_long_run.py come from.

1. tests/golden/long_run_stats.json is the oracle's: its first steps are regenerated here from the seeded inputs.
2. The numbers the GPU test's docstring and DESIGN.md G20 quote are asserted from the committed JSON: how far
   two FP64 oracle runs whose inputs differ by one FP32 ulp drift apart at the configurations' own size.
3. The same experiment is re-run live at 16^3 (seconds): laminar agreement, then chaos -- no FP32 implementation
   can be held to a tighter bar than the oracle holds against itself, and a 64-sample percentile of a chaotic
   flow cannot be held to 10 %.
Nothing here touches the CUDA path."""
import importlib.util
import json
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
_spec = importlib.util.spec_from_file_location("make_long_run_stats",
                                               os.path.join(HERE, "golden", "make_long_run_stats.py"))
G = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(G)
with open(os.path.join(HERE, "golden", "long_run_stats.json")) as _fh:
    GOLD = json.load(_fh)
Q50, Q90 = G.QUANTILES.index(50), G.QUANTILES.index(90)


def _rel(a, b):
    return abs(a - b) / max(abs(a), 1e-300)


def _self_differences(block, key):
    return {r["step"]: _rel(key(r), key(s)) for r, s in zip(block["A"]["checkpoints"], block["B"]["checkpoints"])}


def test_golden_file_is_the_oracles():
    """Shapes are BASELINE.json's, and the first two recorded tracer rows of run A come out of the oracle again
    (2 steps at 32^3: ~2e9 pair evaluations)."""
    import oracle
    c2, c3 = GOLD["config2"], GOLD["config3"]
    assert GOLD["quantiles"] == G.QUANTILES and GOLD["perturb_seed"] == G.PERTURB_SEED
    assert c2["A"]["n"] == 32768 and c2["A"]["steps"] == 1000 and len(c2["A"]["tracer_index"]) == 64
    assert c2["A"]["tracer_index"] == [512 * t for t in range(64)]                       # G18
    assert [r["step"] for r in c2["A"]["checkpoints"]] == G.CHECKPOINTS_2
    assert c3["A"]["n"] == 131072 and c3["A"]["steps"] == 100
    assert [r["step"] for r in c3["A"]["checkpoints"]] == [0] + G.CHECKPOINTS_3
    assert abs(c2["A"]["a_end"] - 1.0) < 2e-6                                            # z = 0 (G12, G13)
    cfg, pm, vel, eps2, tr_idx = G.config2_setup(32)
    st = oracle.State(pm, vel, eps2, cfg.G)
    mids, _ = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, 2)
    rows = np.array(c2["A"]["tracer_rows_first10"])
    for n, (a, H) in enumerate(mids):
        st.step(cfg.tau, a, H)
        got = st.v[tr_idx].astype(np.float32).astype(np.float64)                          # the ring stores FP32
        assert np.abs(got - rows[n]).max() <= 1e-9 * np.abs(rows[n]).max(), n


def test_one_ulp_sensitivity_at_full_size_is_what_the_docs_quote():
    c2, c3 = GOLD["config2"], GOLD["config3"]
    T = _self_differences(c2, lambda r: r["T"])
    W = _self_differences(c2, lambda r: r["W"])
    R = _self_differences(c2, lambda r: r["r_half"])
    q50 = _self_differences(c2, lambda r: r["speed_q"][Q50])
    q90 = _self_differences(c2, lambda r: r["speed_q"][Q90])
    # laminar up to the first collapse (steps 10, 30, 50): the two oracle runs agree to better than 1e-5
    for s in (10, 30, 50):
        assert max(T[s], W[s], R[s], q50[s], q90[s]) < 1e-5, s
    # saturated chaos from step 200 on: 1-2 % on the bulk statistics -- so 1e-3 cannot be asked there, and the
    # GPU test's cap 3 x sat stays below G20's 10 %
    chaotic = [s for s in T if s >= 200]
    sat = {k: max(d[s] for s in chaotic) for k, d in (("T", T), ("W", W), ("r_half", R), ("q50", q50), ("q90", q90))}
    assert 0.015 < sat["T"] < 0.025 and 0.008 < sat["W"] < 0.015 and 0.015 < sat["r_half"] < 0.025
    assert 0.010 < sat["q50"] < 0.020 and 0.010 < sat["q90"] < 0.020
    assert all(3 * v < 0.10 for v in sat.values())
    # ... and inside that regime the pointwise |A - B| of ONE checkpoint is no scale: it is a single draw, and the two
    # runs can cross -- W at step 800 differs by 1.0e-4 between neighbours at 1e-2, T spans a factor 5, r_half 7.
    # The GPU test therefore holds every chaotic checkpoint to 3 x sat, not to 100 x its own pointwise difference
    # (which at such a crossing, 1.03 % for W, would be tighter than what the oracle's two runs differ by elsewhere)
    assert W[800] < 2e-4 and min(W[700], W[900]) > 50 * W[800] and 100 * W[800] < sat["W"]
    for d in (T, W, R, q50):
        assert max(d[s] for s in chaotic) > 4 * min(d[s] for s in chaotic)
    # the 64-tracer percentiles of SURVEY G20: the oracle differs from itself by far more than 10 %
    tm = _self_differences(c2, lambda r: float(np.median(r["tracer_speed"])))
    tp = _self_differences(c2, lambda r: float(np.percentile(r["tracer_speed"], 90)))
    assert max(tm[s] for s in chaotic) > 0.15 and max(tp[s] for s in chaotic) > 0.20
    # ... while, measured in percentile points of the all-particle distribution, A and B stay within 3 sigma of each
    # other, sigma = 6.25 points at the median, 3.75 at p90 per run (two runs differ with sqrt(2) sigma, so this is
    # 2.1 sigma of the difference): the unit the GPU test uses, with 4 sqrt(2) sigma
    for ra, rb in zip(c2["A"]["checkpoints"], c2["B"]["checkpoints"]):
        for q, sigma in ((50, 6.25), (90, 3.75)):
            pa = np.interp(np.percentile(ra["tracer_speed"], q), ra["speed_q"], G.QUANTILES)
            pb = np.interp(np.percentile(rb["tracer_speed"], q), ra["speed_q"], G.QUANTILES)
            assert abs(pa - pb) <= 3.0 * sigma, (ra["step"], q, pa, pb)
    # config 3 stays laminar over its 100 steps
    for key in (lambda r: r["W"], lambda r: r["r_half"], lambda r: r["speed_q"][Q50], lambda r: r["speed_q"][Q90]):
        assert max(_self_differences(c3, key).values()) < 2e-4           # worst: 1.2e-4 (90th speed percentile, step 70)
    assert max(v for s, v in _self_differences(c3, lambda r: r["T"]).items() if s > 0) < 2e-4


def test_chaos_calibration_reproduced_live_at_16_cubed():
    """The experiment behind the thresholds, small enough to run here: config 2 at 16^3, 300 steps, from the
    inputs of record and from inputs moved by one FP32 ulp."""
    checkpoints = [10, 30, 100, 200, 300]
    A = G.run_config2(16, 300, checkpoints, perturbed=False)["checkpoints"]
    B = G.run_config2(16, 300, checkpoints, perturbed=True)["checkpoints"]
    diff = {r["step"]: {"T": _rel(r["T"], s["T"]), "W": _rel(r["W"], s["W"]), "r": _rel(r["r_half"], s["r_half"]),
                        "tp90": _rel(np.percentile(r["tracer_speed"], 90), np.percentile(s["tracer_speed"], 90))}
            for r, s in zip(A, B)}
    for s in (10, 30):                                               # laminar: far inside the GPU test's 1e-3 floor
        assert max(diff[s].values()) < 1e-5, diff[s]
    late = [diff[s] for s in (200, 300)]
    assert max(d["T"] for d in late) > 2e-3                           # chaos: 1e-3 can no longer be asked ...
    assert max(max(d["T"], d["W"], d["r"]) for d in late) < 0.10      # ... but G20's 10 % still can, of the bulk
    assert min(r["r_half"] for r in A) < 0.35 * A[0]["r_half"]       # the box did collapse (G7)
