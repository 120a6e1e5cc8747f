"""Long runs are compared statistically (north_star; reading G20): the paper-shaped run of config 2 --
lattice + small Gaussian displacements, flat LCDM, z = 50 -> 0 in 1000 uniform steps, 64 tracers --
at 16^3 particles so that the FP64 oracle follows all 1000 steps in seconds.  The dynamics are chaotic
(and, with the literal open-boundary eq. (1), the box collapses as a whole near step 280, G7), so beyond
the 10-step window only ensemble quantities are compared: kinetic and potential energy, half-mass radius,
the speed distribution (median and 90th percentile over all particles) and the total power of the
tracer spectra.

With the literal open-boundary eq. (1) the cold box falls onto its centre as a whole (G7): the half-mass
radius shrinks 17 % in the first 10 steps and reaches its minimum near step 50, after which the motion is
chaotic.  Thresholds: 1e-3 while the flow is laminar (steps 10 and 30); 15 % afterwards -- the FP64 oracle
run twice from inputs that differ by one FP32 ulp in each coordinate already differs from itself by up to
3.5 % (T, step 200) and 7.8 % (T, step 900), so nothing tighter can be asked of any FP32 run."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_1208_3444_b200 import binding as B  # noqa: E402
from paper_1208_3444_b200 import inputs  # noqa: E402
from conftest import record_parity  # noqa: E402

SIDE = 16
STEPS = 1000
CHECKPOINTS = [10, 30] + list(range(100, STEPS + 1, 100))


def _half_mass_radius(x, m):
    c = (m[:, None] * x).sum(0) / m.sum()
    return float(np.median(np.linalg.norm(x - c, axis=1)))          # equal masses: median = half-mass


def test_config2_shaped_run_statistics():
    from paper_1208_3444_b200.harness import Session
    cfg, pm, vel = inputs.make_config(2, SIDE ** 3)
    eps2 = np.float32(np.float32(0.05 / SIDE) ** 2)
    tr_idx = (np.arange(64) * (cfg.n // 64)).astype(np.int32)
    m = pm[:, 3].astype(np.float64)

    gpu = []
    with Session(cfg.G, cfg.n) as s:
        s.upload(pm, vel, eps2)
        s.trace(tr_idx, STEPS)
        a, done = cfg.a_start, 0
        for cp in CHECKPOINTS:
            a = s.run_native(cfg.cosmo, a, cfg.tau, cp - done)
            done = cp
            d = s.diagnostics(a, with_potential=True)
            pos, v = s.download()
            gpu.append((a, d[7], d[8], _half_mass_radius(pos[:, :3].astype(np.float64), m),
                        np.linalg.norm(v[:, :3].astype(np.float64), axis=1)))
        spec_gpu = s.trace_spectrum(0, STEPS)
        rows_gpu = s.trace_read(0, STEPS)
    assert a == pytest.approx(1.0, abs=2e-6)                          # z = 0 reached (tau of G13)

    st = oracle.State(pm, vel, eps2, cfg.G)
    mids, ends = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, STEPS)
    ref, rows_ref = [], np.zeros((STEPS, 64, 4), dtype=np.float32)
    for n, (am, Hm) in enumerate(mids):
        st.step(cfg.tau, am, Hm)
        rows_ref[n, :, :3] = st.v[tr_idx]
        if (n + 1) in CHECKPOINTS:
            d = st.diagnostics(ends[n + 1], with_potential=True)
            ref.append((ends[n + 1], d[7], d[8], _half_mass_radius(st.x, m), np.linalg.norm(st.v, axis=1)))

    worst = {"T": 0.0, "W": 0.0, "r_half": 0.0}
    early = {"T": 0.0, "W": 0.0, "r_half": 0.0}
    for step, g, r in zip(CHECKPOINTS, gpu, ref):
        tol = 1e-3 if step <= 30 else 0.15
        assert g[0] == pytest.approx(r[0], rel=1e-8)
        for name, i in (("T", 1), ("W", 2), ("r_half", 3)):
            rel = abs(g[i] - r[i]) / abs(r[i])
            worst[name] = max(worst[name], rel)
            if step <= 30:
                early[name] = max(early[name], rel)
            assert rel <= tol, (step, name, g[i], r[i])
        if step in (100, 500, 1000):
            for q in (50, 90):
                pg, pr = np.percentile(g[4], q), np.percentile(r[4], q)
                assert abs(pg - pr) <= 0.15 * pr, (step, q, pg, pr)
    record_parity("1000-step config-2-shaped run (16^3)", **{"worst_rel_" + k: v for k, v in worst.items()},
                  **{"laminar_rel_" + k: v for k, v in early.items()})

    # the run is not trivial: the box collapses onto its centre (G7) and the kinetic energy grows several-fold
    radii = [r[3] for r in ref]
    assert min(radii) < 0.1 * radii[0] and max(r[1] for r in ref) > 3 * ref[0][1]

    # tracer spectra: total power (Parseval: = sum_s |v|^2) per tracer, summed over the 64 tracers
    spec_ref = oracle.trace_spectrum(rows_ref)
    assert np.abs(spec_gpu - oracle.trace_spectrum(rows_gpu)).max() <= 1e-10 * spec_gpu.max()
    assert spec_gpu.sum() == pytest.approx(spec_ref.sum(), rel=0.15)
    # the first 10 recorded steps still agree sample by sample
    vr = np.sqrt((rows_ref[:10, :, :3].astype(np.float64) ** 2).sum(2).mean())
    assert np.abs(rows_gpu[:10, :, :3] - rows_ref[:10, :, :3]).max() <= 2e-4 * vr


def test_config3_shaped_cold_collapse_energy_and_virial():
    """Config 3's own long run (reading G13/G20): Plummer sphere + 30 % background, cold start, static
    background, 100 steps of tau = 1e-3 through maximum compression (near step 50) to a virialised state --
    at N = 8192 so the oracle follows it in seconds.  Static limit: T + W is conserved by the flow, so the
    GPU run is held to an absolute energy budget, and T, W are compared with the oracle's."""
    from paper_1208_3444_b200.harness import Session
    cfg, pm, vel = inputs.make_config(3, 8192)
    steps, every = 100, 10
    gpu = []
    with Session(cfg.G, cfg.n) as s:
        s.upload(pm, vel, cfg.eps2)
        d = s.diagnostics(1.0, with_potential=True)
        gpu.append((d[7], d[8]))
        for _ in range(steps // every):
            s.run_native(None, 1.0, cfg.tau, every)
            d = s.diagnostics(1.0, with_potential=True)
            gpu.append((d[7], d[8]))
            assert np.abs(d[1:4]).max() <= 1e-5 * np.sqrt(2 * d[7] * d[0] + 1e-30) + 1e-9     # sum m v stays ~0
    st = oracle.State(pm, vel, cfg.eps2, cfg.G)
    d = st.diagnostics(1.0, with_potential=True)
    ref = [(d[7], d[8])]
    for n in range(steps):
        st.step(cfg.tau, 1.0, 0.0)
        if (n + 1) % every == 0:
            d = st.diagnostics(1.0, with_potential=True)
            ref.append((d[7], d[8]))
    E0 = ref[0][0] + ref[0][1]
    assert gpu[0][0] == 0.0 and gpu[0][1] == pytest.approx(ref[0][1], rel=1e-6)
    drift_gpu = max(abs(T + W - E0) / abs(E0) for T, W in gpu)
    drift_ref = max(abs(T + W - E0) / abs(E0) for T, W in ref)
    worst = 0.0
    for k, ((Tg, Wg), (Tr, Wr)) in enumerate(zip(gpu, ref)):
        if k == 0:
            continue
        tol = 1e-3 if k <= 3 else 1e-2                    # measured 5.5e-5 over the whole run
        worst = max(worst, abs(Tg - Tr) / Tr, abs(Wg - Wr) / abs(Wr))
        assert abs(Tg - Tr) <= tol * Tr and abs(Wg - Wr) <= tol * abs(Wr), (k * every, Tg, Tr, Wg, Wr)
    record_parity("100-step config-3-shaped run (N=8192)", energy_drift_gpu=drift_gpu, energy_drift_oracle=drift_ref,
                  worst_rel_T_or_W=worst)
    assert drift_gpu <= max(2.0 * drift_ref, 0.02)
    assert max(T for T, _ in ref) > 0.5 * abs(ref[0][1])   # it did collapse: T reaches the scale of |W0|
