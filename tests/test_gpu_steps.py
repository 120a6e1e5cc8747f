"""T2/T3 (trajectories): eqs. (3)-(5) on the GPU against the FP64 oracle, through the C ABI.

north_star: "Trajectories after 10 steps must agree to relative position error <= 1e-5", read as
max_k |x_gpu,k - x_ref,k| / L_box <= 1e-5 with L_box = 1 (reading G16), with the guard that the
reference itself moved >= 100 x the tolerance, so a no-op integrator cannot pass.
The GPU side takes a, H from libcolatus' host Friedmann helpers, the oracle from its own RK4.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_1208_3444_b200 import binding as B  # noqa: E402
from paper_1208_3444_b200 import inputs  # noqa: E402
from conftest import record_parity  # noqa: E402

POS_TOL = 1e-5


def _session(G, n):
    from paper_1208_3444_b200.harness import Session
    return Session(G, n)


def _oracle_run(cfg, pm, vel, steps):
    st = oracle.State(pm, vel, cfg.eps2, cfg.G)
    mids, ends = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, steps)
    for a, H in mids:
        st.step(cfg.tau, a, H)
    return st, mids, ends


@pytest.mark.parametrize("index", [1, 2, 3])
def test_ten_step_trajectory_parity(index):
    cfg, pm, vel = inputs.make_config(index)
    steps = cfg.parity_steps
    with _session(cfg.G, cfg.n) as s:
        s.upload(pm, vel, cfg.eps2)
        if cfg.n_tracers:
            s.trace(inputs.tracer_indices(cfg), steps)
        a_end = s.run(cfg.cosmo, cfg.a_start, cfg.tau, steps)
        pos, v = s.download()
        diag = s.diagnostics(a_end)
        tr = s.trace_read(0, steps) if cfg.n_tracers else None
    st, mids, ends = _oracle_run(cfg, pm, vel, steps)
    x0 = pm[:, :3].astype(np.float64)
    moved = np.linalg.norm(st.x - x0, axis=1).max()
    assert moved >= 100 * POS_TOL, f"vacuous: reference moved only {moved:g}"          # G16 guard
    err = np.linalg.norm(pos[:, :3].astype(np.float64) - st.x, axis=1).max()
    record_parity(f"{steps}-step trajectory config {index}", n=cfg.n, max_dx_over_box=err, ref_moved=moved)
    assert err <= POS_TOL, (index, err)
    assert a_end == pytest.approx(ends[-1], rel=1e-9)
    assert np.array_equal(pos[:, 3], pm[:, 3])                                          # masses untouched
    # velocities: relative to the rms speed
    vrms = np.sqrt((st.v ** 2).sum(1).mean())
    assert np.linalg.norm(v[:, :3].astype(np.float64) - st.v, axis=1).max() <= 2e-4 * vrms
    # diagnostics against the oracle's
    dref = st.diagnostics(ends[-1])
    assert diag[0] == pytest.approx(dref[0], rel=1e-7)
    assert diag[7] == pytest.approx(dref[7], rel=1e-4)
    assert np.allclose(diag[9:12], dref[9:12], atol=1e-6)
    assert diag[12] == steps
    if tr is not None:
        idx = inputs.tracer_indices(cfg)
        assert np.array_equal(tr[-1, :, :3], v[idx, :3])                                 # ring = v^{n+1}
        assert np.allclose(tr[-1, :, 3], mids[-1][0], rtol=1e-6)                         # tag = a (G18)
        st5, _, _ = _oracle_run(cfg, pm, vel, 5)
        assert np.linalg.norm(tr[4, :, :3].astype(np.float64) - st5.v[idx], axis=1).max() <= 2e-4 * vrms


def test_momentum_law_every_step():
    """P9 on the GPU: P^{n+1} = cv_n P^n (sum m F = 0), any configuration, per step."""
    cfg, pm, vel = inputs.make_config(1)
    rng = np.random.Generator(np.random.PCG64(5))
    vel = vel.copy()
    vel[:, :3] = 0.3 * rng.normal(size=(cfg.n, 3)).astype(np.float32) + np.float32(0.5)
    with _session(cfg.G, cfg.n) as s:
        s.upload(pm, vel, cfg.eps2)
        a = cfg.a_start
        P = s.diagnostics(a)[1:4]
        for _ in range(5):
            a_mid = B.colatus_a_advance(cfg.cosmo, a, 0.5 * cfg.tau)
            H = B.colatus_hubble(cfg.cosmo, a_mid)
            B.colatus_step(cfg.tau, a_mid, H)
            a = B.colatus_a_advance(cfg.cosmo, a_mid, 0.5 * cfg.tau)
            Pn = s.diagnostics(a)[1:4]
            cv = (1 - H * cfg.tau) / (1 + H * cfg.tau)
            assert np.allclose(Pn, cv * P, rtol=2e-5, atol=2e-6 * np.abs(P).max())
            P = Pn


def test_static_energy_conservation_and_potential():
    """P8 on the GPU: a=1, H=0 -> T+W conserved; W from the potential-fused force pass (eq. 7)."""
    cfg, pm, vel = inputs.make_config(3, n_override=8192)
    with _session(cfg.G, cfg.n) as s:
        s.upload(pm, vel, cfg.eps2)
        d0 = s.diagnostics(1.0, True)
        s.run(None, 1.0, cfg.tau, 10)
        d1 = s.diagnostics(1.0, True)
    st = oracle.State(pm, vel, cfg.eps2, cfg.G)
    r0 = st.diagnostics(1.0, True)
    assert d0[8] == pytest.approx(r0[8], rel=2e-6)                    # W
    assert d0[7] == 0.0
    E0, E1 = d0[7] + d0[8], d1[7] + d1[8]
    assert abs(E1 - E0) <= 2e-5 * abs(E0)
    assert d1[7] > 1e-4 * abs(E0)                                      # something happened


def test_layzer_irvine_on_the_gpu():
    """P11 on the GPU (tier T3): with T = 1/2 sum m a^2 v^2 and W from the potential-fused force pass,
    eqs. (1), (3)-(5) and (7) imply d(T+W)/dt = -H (2T + W).  Config 1 (EdS), a fixed time span covered in 40 and
    in 80 steps, colatus_diagnostics(with_potential) at every step end: the trapezoid-integrated residual is far
    below |Delta E| and shrinks ~4x when tau halves (the scheme is second order), and T, W follow the oracle's."""
    cfg, pm, vel = inputs.make_config(1)
    span = 0.004
    res, dE = [], []
    for steps in (40, 80):
        tau = span / steps
        mids, ends = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, tau, steps)
        st = oracle.State(pm, vel, cfg.eps2, cfg.G)
        with _session(cfg.G, cfg.n) as s:
            s.upload(pm, vel, cfg.eps2)
            d = s.diagnostics(ends[0], True)
            E = [d[7] + d[8]]
            rhs = [B.colatus_hubble(cfg.cosmo, ends[0]) * (2 * d[7] + d[8])]
            a = cfg.a_start
            for i in range(steps):
                a_mid = B.colatus_a_advance(cfg.cosmo, a, 0.5 * tau)
                B.colatus_step(tau, a_mid, B.colatus_hubble(cfg.cosmo, a_mid))
                a = B.colatus_a_advance(cfg.cosmo, a_mid, 0.5 * tau)
                assert a == pytest.approx(ends[i + 1], rel=1e-9)
                d = s.diagnostics(a, True)
                E.append(d[7] + d[8])
                rhs.append(B.colatus_hubble(cfg.cosmo, a) * (2 * d[7] + d[8]))
                st.step(tau, *mids[i])
                r = st.diagnostics(ends[i + 1], True)
                assert d[8] == pytest.approx(r[8], rel=1e-4), (steps, i)
                assert abs(d[7] - r[7]) <= 1e-4 * abs(r[8]), (steps, i)        # T starts at 0: scale by |W|
        rhs = np.array(rhs)
        integral = tau * (rhs.sum() - 0.5 * (rhs[0] + rhs[-1]))                # trapezoid
        res.append(abs(E[-1] - E[0] + integral))
        dE.append(abs(E[-1] - E[0]))
        assert res[-1] <= 1e-2 * dE[-1], (steps, res, dE)
    record_parity("Layzer-Irvine on the GPU (config 1, 40 / 80 steps)", residual_40=res[0], residual_80=res[1],
                  delta_E=dE[1])
    assert res[0] / res[1] == pytest.approx(4.0, rel=0.35), res


def test_step_coeffs_equals_step_and_is_reproducible():
    cfg, pm, vel = inputs.make_config(1)
    out = []
    for mode in ("step", "coeffs", "split"):
        with _session(cfg.G, cfg.n) as s:
            s.upload(pm, vel, cfg.eps2)
            tau, a, H = cfg.tau, 0.03, 11.0
            for _ in range(3):
                if mode == "step":
                    B.colatus_step(tau, a, H)
                elif mode == "coeffs":
                    B.colatus_step_coeffs(*B.colatus_step_coefficients(tau, a, H))
                else:
                    d1, cv, ck, d2 = B.colatus_step_coefficients(tau, a, H)
                    B.colatus_drift(d1)
                    B.colatus_force_kick_drift(cv, ck, d2)
            out.append(s.download())
    for pos, v in out[1:]:
        assert np.array_equal(pos, out[0][0]) and np.array_equal(v, out[0][1])


def test_trace_ring_wraps():
    cfg, pm, vel = inputs.make_config(1)
    idx = np.array([5, 4095, 0, 77], dtype=np.int32)
    with _session(cfg.G, cfg.n) as s:
        s.upload(pm, vel, cfg.eps2)
        s.trace(idx, 4)
        vs = []
        for k in range(6):
            B.colatus_step(cfg.tau, 0.05, 3.0)
            vs.append(s.download()[1][idx, :3])
        got = s.trace_read(2, 4)                      # steps 2..5 live in slots 2,3,0,1
        for j in range(4):
            assert np.array_equal(got[j, :, :3], vs[2 + j])
        with pytest.raises(B.ColatusError):
            s.trace_read(1, 2)                        # step 1 was overwritten
        with pytest.raises(B.ColatusError):
            s.trace_read(5, 2)                        # step 6 not taken yet


def test_target_range_stepping_matches_full():
    """Two half ranges stepped one after the other on shared arrays reproduce the full step up to the summation
    order (the source split is chosen per target count, reading G14: FP32 sums differ at the 1e-6 level between
    tilings) -- the single-GPU emulation of the target-sharded multi-GPU step."""
    import torch
    cfg, pm, vel = inputs.make_config(1)
    with _session(cfg.G, cfg.n) as s:
        s.upload(pm, vel, cfg.eps2)
        B.colatus_step(cfg.tau, 0.05, 3.0)
        full_pos, full_vel = s.download()
        s.upload(pm, vel, cfg.eps2)
        d1, cv, ck, d2 = B.colatus_step_coefficients(cfg.tau, 0.05, 3.0)
        h = cfg.n // 2
        for b in (0, h):
            B.colatus_set_target_range(b, h)
            B.colatus_drift(d1)
        snapshot = s.pos.clone()                       # all-gathered half-step positions
        new_pos = []
        acc_half = torch.zeros((h, 4), dtype=torch.float32, device=s.device)
        for b in (0, h):
            s.pos.copy_(snapshot)
            B.colatus_upload(s.pos, s.vel, acc_half, cfg.n, cfg.eps2)
            B.colatus_set_target_range(b, h)
            B.colatus_force_kick_drift(cv, ck, d2)
            new_pos.append(s.pos[b:b + h].clone())
        B.colatus_set_target_range(0, cfg.n)
        pos, v = s.download()
        pos[:h] = new_pos[0].cpu().numpy()
        pos[h:] = new_pos[1].cpu().numpy()
    v_rms = float(np.sqrt((full_vel[:, :3].astype(np.float64) ** 2).sum(1).mean()))
    assert np.abs(pos - full_pos).max() <= 1e-7 and np.abs(v - full_vel).max() <= 2e-6 * v_rms


@pytest.mark.parametrize("index,n_override", [(1, None), (3, 100), (3, 20000)])
def test_fused_step_equals_separate_kernels_bitwise(index, n_override):
    """colatus_step_coeffs takes the fused route (drift+staging, force, reduce+kick+drift); colatus_drift +
    colatus_force_kick_drift take the separate kernels.  Same arithmetic, statement for statement: positions,
    velocities, the acc buffer and the tracer ring must agree to the bit (single- and multi-split sizes)."""
    cfg, pm, vel = inputs.make_config(index, n_override)
    rng = np.random.Generator(np.random.PCG64(3))
    vel = vel.copy()
    vel[:, :3] = 0.02 * rng.standard_normal((cfg.n, 3)).astype(np.float32)
    tr = np.arange(0, cfg.n, max(cfg.n // 8, 1), dtype=np.int32)[:8]
    coeffs = [(0.4e-3, 0.9, 1.1e-3, 0.6e-3), (0.5e-3, 1.0, 0.7e-3, 0.5e-3), (0.3e-3, 0.8, 2.0e-3, 0.2e-3)]
    outs = []
    for fused in (True, False):
        with _session(cfg.G, cfg.n) as s:
            s.upload(pm, vel, cfg.eps2)
            s.trace(tr, 2)
            for d1, cv, ck, d2 in coeffs:
                if fused:
                    B.colatus_step_coeffs(d1, cv, ck, d2)
                else:
                    B.colatus_drift(d1)
                    B.colatus_force_kick_drift(cv, ck, d2)
            pos, v = s.download()
            outs.append((pos, v, s.acc.cpu().numpy(), s.ring.cpu().numpy(), s.diagnostics(1.0)[12]))
    for a, b in zip(outs[0], outs[1]):
        assert np.array_equal(a, b)
    assert outs[0][4] == len(coeffs)
