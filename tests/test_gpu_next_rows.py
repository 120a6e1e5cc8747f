"""GPU parity for the NEXT rows of SURVEY 8f against the FP64 oracle, through the C ABI:
f1 symplectic step of eq. (9), f2 deformation source of eq. (10),
f5 mean-density background term (reading G22).  Tolerances as for the main path (G16, G17)."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_1208_3444_b200 import binding as B  # noqa: E402
from paper_1208_3444_b200 import inputs  # noqa: E402

POS_TOL, MEDIAN_TOL, MAX_TOL = 1e-5, 1e-5, 1e-4


def _session(G, n):
    from paper_1208_3444_b200.harness import Session
    return Session(G, n)


def _force_errors(acc_gpu, acc_ref):
    d = np.linalg.norm(acc_gpu.astype(np.float64) - acc_ref, axis=1)
    nr = np.linalg.norm(acc_ref, axis=1)
    return float(np.median(d / nr)), float(d.max() / np.sqrt((nr ** 2).mean()))


@pytest.mark.parametrize("index", [1, 2])
def test_symplectic_ten_step_parity_and_momentum(index):
    """Eq. (9): 10 D-K-D steps in w = a^2 v.  Positions within 1e-5 of the box of the oracle's; the
    canonical momentum sum m w is conserved (cv = 1 and sum m F = 0), unlike eqs. (3)-(5)."""
    cfg, pm, vel = inputs.make_config(index)
    rng = np.random.Generator(np.random.PCG64(50 + index))
    w0 = vel.copy()
    w0[:, :3] = (cfg.a_start ** 2) * 0.05 * rng.standard_normal((cfg.n, 3)).astype(np.float32)
    steps = 10
    with _session(cfg.G, cfg.n) as s:
        s.upload(pm, w0, cfg.eps2)
        s.trace(np.arange(0, cfg.n, cfg.n // 16, dtype=np.int32), steps)
        a = cfg.a_start
        for _ in range(steps):
            a = B.colatus_step_symplectic(cfg.cosmo, a, cfg.tau)
        pos, w = s.download()
        diag = s.diagnostics(1.0)
        tr = s.trace_read(0, steps)
    st = oracle.State(pm, w0, cfg.eps2, cfg.G)
    a_ref = cfg.a_start
    for _ in range(steps):
        a_ref = st.step_symplectic(cfg.cosmo, a_ref, cfg.tau)
    assert a == pytest.approx(a_ref, rel=1e-9)
    moved = np.linalg.norm(st.x - pm[:, :3].astype(np.float64), axis=1).max()
    assert moved >= 100 * POS_TOL, moved
    err = np.linalg.norm(pos[:, :3].astype(np.float64) - st.x, axis=1).max()
    assert err <= POS_TOL, (index, err)
    wrms = np.sqrt((st.v ** 2).sum(1).mean())
    assert np.linalg.norm(w[:, :3].astype(np.float64) - st.v, axis=1).max() <= 2e-4 * wrms
    m = pm[:, 3].astype(np.float64)
    P0 = (m[:, None] * w0[:, :3].astype(np.float64)).sum(0)
    scale = (m[:, None] * np.abs(w[:, :3].astype(np.float64))).sum()
    assert np.abs(np.array(diag[1:4]) - P0).max() <= 3e-6 * scale
    assert np.allclose(tr[-1, :, 3], a, rtol=1e-6)                      # tag = a(t + tau)
    assert np.array_equal(tr[-1, :, :3], w[::cfg.n // 16, :3])


def test_symplectic_step_equals_step_coeffs_bitwise():
    cfg, pm, vel = inputs.make_config(1)
    outs = []
    for mode in (0, 1):
        with _session(cfg.G, cfg.n) as s:
            s.upload(pm, vel, cfg.eps2)
            a = cfg.a_start
            for _ in range(3):
                if mode == 0:
                    a = B.colatus_step_symplectic(cfg.cosmo, a, cfg.tau)
                else:
                    d1, cv, ck, d2, a = B.colatus_symplectic_coefficients(cfg.cosmo, a, cfg.tau)
                    B.colatus_step_coeffs(d1, cv, ck, d2)
            outs.append(s.download())
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


def test_deformation_and_background_forces():
    """Eq. (10) source and the background term appear in colatus_forces / forces_range, and switch off."""
    cfg, pm, _ = inputs.make_config(3, n_override=20000)
    xpsi, S = np.array([0.45, 0.55, 0.5]), 0.4
    cen, rho = np.array([0.5, 0.5, 0.5]), 1.0
    tg = np.arange(0, 20000, 7)
    x = pm[:, :3].astype(np.float64)
    with _session(2.0, cfg.n) as s:
        base = s.forces(pm, cfg.eps2).cpu().numpy()
        B.colatus_set_deformation(xpsi, S)
        f_def = s.forces(pm, cfg.eps2).cpu().numpy()
        B.colatus_set_background(cen, rho)
        f_both = s.forces(pm, cfg.eps2, potential=True).cpu().numpy()
        f_rng = s.forces(pm, cfg.eps2, target_range=(5000, 3001)).cpu().numpy()
        B.colatus_set_deformation(None, 0.0)
        f_bg = s.forces(pm, cfg.eps2).cpu().numpy()
        B.colatus_set_background(None, 0.0)
        again = s.forces(pm, cfg.eps2).cpu().numpy()
    assert np.array_equal(base, again)
    ref0 = oracle.forces(pm, cfg.eps2, 2.0, tg)
    for got, d, b in ((f_def, (xpsi, S), None), (f_both, (xpsi, S), (cen, rho)), (f_bg, None, (cen, rho))):
        ref = oracle.add_external(x, ref0.copy(), cfg.eps2, 2.0, targets=tg, deformation=d, background=b)
        med, mx = _force_errors(got[tg, :3], ref)
        assert med <= MEDIAN_TOL and mx <= MAX_TOL, (med, mx)
        assert np.abs(ref - ref0).max() > 1e3 * MAX_TOL * np.sqrt((ref0 ** 2).sum(1).mean())   # non-vacuous
    # a target range picks its own source-split geometry, so it is close to, not bitwise equal to, the full
    # run (G14); it is checked against the oracle in its own right
    rt = np.arange(5000, 8001)
    ref_r = oracle.add_external(x, oracle.forces(pm, cfg.eps2, 2.0, rt), cfg.eps2, 2.0, targets=rt,
                                deformation=(xpsi, S), background=(cen, rho))
    med, mx = _force_errors(f_rng[:, :3], ref_r)
    assert med <= MEDIAN_TOL and mx <= MAX_TOL, (med, mx)
    sc = np.sqrt((ref_r ** 2).sum(1).mean())
    assert np.abs(f_rng[:, :3] - f_both[5000:8001, :3]).max() <= 1e-5 * sc
    # the external terms are not part of acc.w (the potential of eq. (1))
    _, phi = oracle.forces(pm, cfg.eps2, 2.0, tg, potential=True)
    assert np.allclose(f_both[tg, 3], phi, rtol=2e-5)


def test_step_with_external_terms_parity():
    cfg, pm, vel = inputs.make_config(1)
    xpsi, S = np.array([0.5, 0.5, 1.5]), 0.5
    cen, rho = np.array([0.5, 0.5, 0.5]), 1.0          # box mean density (total mass 1 in unit box)
    steps = 10
    with _session(cfg.G, cfg.n) as s:
        B.colatus_set_deformation(xpsi, S)
        B.colatus_set_background(cen, rho)
        s.upload(pm, vel, cfg.eps2)
        s.run(cfg.cosmo, cfg.a_start, cfg.tau, steps)
        pos, _ = s.download()
    st = oracle.State(pm, vel, cfg.eps2, cfg.G)
    st.deformation, st.background = (xpsi, S), (cen, rho)
    mids, _ = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, steps)
    for a, H in mids:
        st.step(cfg.tau, a, H)
    plain = oracle.State(pm, vel, cfg.eps2, cfg.G)
    for a, H in mids:
        plain.step(cfg.tau, a, H)
    assert np.linalg.norm(st.x - plain.x, axis=1).max() >= 100 * POS_TOL          # the terms matter
    assert np.linalg.norm(pos[:, :3].astype(np.float64) - st.x, axis=1).max() <= POS_TOL


def test_external_argument_validation():
    cfg, pm, _ = inputs.make_config(1)
    with _session(1.0, cfg.n):
        for fn in (B.colatus_set_deformation, B.colatus_set_background):
            with pytest.raises(B.ColatusError):
                fn((0.0, 0.0, 0.0), float("nan"))
            with pytest.raises(B.ColatusError):
                fn((0.0, float("inf"), 0.0), 1.0)
            assert getattr(B.lib(), fn.__name__)(None, 1.0) == B.INVALID_ARG
        with pytest.raises(B.ColatusError):
            B.colatus_step_symplectic(cfg.cosmo, 0.5, 1e-3)                       # not uploaded
