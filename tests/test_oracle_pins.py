"""T0: pin the CPU oracle to what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path: every expected
value is a closed form, an exact rational worked example (tests/golden/), an invariant,
or an independent few-line NumPy evaluation on tiny inputs.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_1208_3444_b200.inputs import Cosmology

RNG = np.random.Generator(np.random.PCG64(12345))


# ----------------------------------------------------------------------------- P1
def test_two_body_closed_form_and_direction():
    """|F on 1| = G m2 r / (r^2+eps^2)^{3/2}, pointing from body 1 TOWARD body 2 (G1)."""
    G, eps2 = 2.5, 0.09
    x = np.array([[0.1, -0.2, 0.3], [0.7, 0.4, -0.5]])
    m = np.array([3.0, 5.0])
    d = x[1] - x[0]
    r = np.linalg.norm(d)
    F = oracle.forces_xm(x, m, eps2, G)
    assert np.allclose(F[0], G * m[1] * r / (r * r + eps2) ** 1.5 * d / r, rtol=1e-14)
    assert np.allclose(F[1], -G * m[0] * r / (r * r + eps2) ** 1.5 * d / r, rtol=1e-14)
    assert np.dot(F[0], d) > 0 and np.dot(F[1], d) < 0           # attraction


def test_softened_force_maximum():
    """max_r G m r/(r^2+eps^2)^{3/2} = 2 G m / (3 sqrt(3) eps^2) at r = eps/sqrt(2)."""
    G, mass, eps = 1.0, 2.0, 0.25
    rs = np.linspace(0.01, 1.0, 2001)
    f = []
    for r in rs:
        F = oracle.forces_xm(np.array([[0, 0, 0], [r, 0, 0.0]]), np.array([0.0, mass]), eps * eps, G)
        f.append(F[0, 0])
    f = np.array(f)
    i = int(np.argmax(f))
    assert abs(rs[i] - eps / math.sqrt(2)) < 1e-3
    fmax = oracle.forces_xm(np.array([[0, 0, 0], [eps / math.sqrt(2), 0, 0.0]]),
                            np.array([0.0, mass]), eps * eps, G)[0, 0]
    assert fmax == pytest.approx(2 * G * mass / (3 * math.sqrt(3) * eps * eps), rel=1e-14)


def _read_golden(path):
    rows = {}
    with open(path) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            tok = line.split()
            rows[tok[0]] = tok[1:]
    return rows


def test_three_body_exact_rational(golden_dir):
    rows = _read_golden(os.path.join(golden_dir, "three_body_rational.txt"))
    x = np.array([[0, 0, 0], [1, 2, 2], [2, 4, 0]], dtype=np.float64)
    m = np.array([1.0, 2.0, 3.0])
    F = oracle.forces_xm(x, m, 16.0, 1.0)
    for i, body in enumerate("ABC"):
        want = [float(Fraction(s)) for s in rows[body]]
        assert np.allclose(F[i], want, rtol=0, atol=2e-17), (body, F[i], want)
    assert np.allclose((m[:, None] * F).sum(axis=0), 0.0, atol=1e-16)


# ----------------------------------------------------------------------------- P2
@pytest.mark.parametrize("n", [2, 17, 500])
def test_newton_third_law(n):
    x = RNG.random((n, 3))
    m = RNG.random(n) + 0.1
    F = oracle.forces_xm(x, m, 1e-4, 1.7)
    num = np.linalg.norm((m[:, None] * F).sum(axis=0))
    den = (m * np.linalg.norm(F, axis=1)).sum()
    assert num / den < 1e-13


# ----------------------------------------------------------------------------- P3
def _fibonacci_shell(n, R):
    i = np.arange(n) + 0.5
    z = 1.0 - 2.0 * i / n
    phi = math.pi * (1.0 + math.sqrt(5.0)) * i
    s = np.sqrt(1.0 - z * z)
    return R * np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def _shell_force_radial(G, M, R, r, eps2):
    """-d/dr of phi(r) = -(G M / 2 r R) [sqrt((R+r)^2+eps^2) - sqrt((R-r)^2+eps^2)]."""
    A = math.sqrt((R + r) ** 2 + eps2)
    B = math.sqrt((R - r) ** 2 + eps2)
    return (G * M / (2 * R)) * (((R + r) / A + (R - r) / B) / r - (A - B) / (r * r))


def _shell_potential(G, M, R, r, eps2):
    return -(G * M / (2 * r * R)) * (math.sqrt((R + r) ** 2 + eps2) - math.sqrt((R - r) ** 2 + eps2))


@pytest.mark.parametrize("eps", [0.001, 0.05, 0.3])
def test_shell_theorem_softened_closed_form(eps):
    G, M, R, n = 1.3, 2.0, 1.0, 10_000
    shell = _fibonacci_shell(n, R)
    direction = np.array([0.36, -0.48, 0.8])                       # unit vector
    tol = {0.1: 3e-6, 0.5: 1.2e-5, 0.8: 9e-5, 1.5: 1.2e-5, 3.0: 3e-7}
    for r, t in tol.items():
        x = np.concatenate([shell, (r * direction)[None, :]], axis=0)
        m = np.concatenate([np.full(n, M / n), [0.0]])
        F, phi = oracle.forces_xm(x, m, eps * eps, G, targets=np.array([n]), potential=True)
        Fr = float(F[0] @ direction)
        Ft = np.linalg.norm(F[0] - Fr * direction)
        scale = G * M / R ** 2
        assert abs(Fr - _shell_force_radial(G, M, R, r, eps * eps)) < t * scale, (r, eps)
        assert Ft < t * scale
        assert abs(phi[0] - _shell_potential(G, M, R, r, eps * eps)) < 10 * t * G * M / R
    # epsilon -> 0 limits: zero inside, G M / r^2 outside
    if eps == 0.001:
        x = np.concatenate([shell, (0.3 * direction)[None, :]], axis=0)
        m = np.concatenate([np.full(n, M / n), [0.0]])
        F = oracle.forces_xm(x, m, eps * eps, G, targets=np.array([n]))
        assert np.linalg.norm(F[0]) < 1e-5 * G * M
        x[-1] = 2.0 * direction
        F = oracle.forces_xm(x, m, eps * eps, G, targets=np.array([n]))
        assert float(F[0] @ direction) == pytest.approx(-G * M / 4.0, rel=1e-5)


# ----------------------------------------------------------------------------- P4
def _numpy_pairwise(x, m, eps2, G):
    """Independent evaluation: full pairwise tensors, diagonal removed by masking."""
    d = x[None, :, :] - x[:, None, :]                 # d[k, j] = x_j - x_k
    s = (d ** 2).sum(-1) + eps2
    w = m[None, :] * s ** -1.5
    np.fill_diagonal(w, 0.0)
    F = G * (w[:, :, None] * d).sum(axis=1)
    p = m[None, :] * s ** -0.5
    np.fill_diagonal(p, 0.0)
    return F, -G * p.sum(axis=1)


@pytest.mark.parametrize("n", [2, 3, 5, 8, 64])
def test_brute_force_tiny_n(n):
    x = RNG.normal(size=(n, 3))
    m = RNG.random(n) + 0.05
    F, phi = oracle.forces_xm(x, m, 0.01, 0.7, potential=True)
    Fw, pw = _numpy_pairwise(x, m, 0.01, 0.7)
    assert np.allclose(F, Fw, rtol=1e-12, atol=1e-14)
    assert np.allclose(phi, pw, rtol=1e-12)


def test_target_list_and_self_skip():
    n = 40
    x = RNG.random((n, 3))
    m = RNG.random(n)
    Fw, _ = _numpy_pairwise(x, m, 1e-3, 1.0)
    tg = np.array([39, 0, 7, 7, 21])
    F = oracle.forces_xm(x, m, 1e-3, 1.0, targets=tg)
    assert np.allclose(F, Fw[tg], rtol=1e-12)
    # two distinct particles at the same place contribute nothing to each other (G4)
    x2 = x.copy()
    x2[1] = x2[0]
    F2 = oracle.forces_xm(x2, m, 1e-3, 1.0)
    x3 = np.delete(x2, 1, axis=0)
    m3 = np.delete(m, 1)
    F3 = oracle.forces_xm(x3, m3, 1e-3, 1.0)
    assert np.allclose(F2[0], F3[0], rtol=1e-12)


def test_float32_entry_promotes_exactly():
    pm = RNG.random((33, 4)).astype(np.float32)
    F = oracle.forces(pm, np.float32(0.01) ** 2, 1.0)
    Fw, _ = _numpy_pairwise(pm[:, :3].astype(np.float64), pm[:, 3].astype(np.float64),
                            float(np.float32(0.01) ** 2), 1.0)
    assert np.allclose(F, Fw, rtol=1e-12)


# ----------------------------------------------------------------------------- P5
def test_symmetries():
    n = 200
    x = RNG.random((n, 3))
    m = RNG.random(n) + 0.1
    eps2, G = 4e-4, 1.0
    F = oracle.forces_xm(x, m, eps2, G)
    perm = RNG.permutation(n)
    assert np.allclose(oracle.forces_xm(x[perm], m[perm], eps2, G), F[perm], rtol=1e-11, atol=1e-13)
    # translation invariance: a general shift moves every coordinate by <= 1 ulp(4) = 9e-16, i.e. <= 1e-12 of
    # the closest separations here, so the forces agree to ~1e-11; a dyadic shift of dyadic inputs is exact
    assert np.allclose(oracle.forces_xm(x + np.array([4.0, -3.7, 1.3]), m, eps2, G), F, rtol=1e-9, atol=1e-12)
    xs = np.round(x * 2 ** 20) / 2 ** 20                                   # translation by 2^k is exact
    assert np.array_equal(oracle.forces_xm(xs + 2.0, m, eps2, G), oracle.forces_xm(xs, m, eps2, G))
    lam = 3.0
    assert np.allclose(oracle.forces_xm(lam * x, m, lam * lam * eps2, G), F / lam ** 2, rtol=1e-12)
    assert np.allclose(oracle.forces_xm(x, 2.5 * m, eps2, G), 2.5 * F, rtol=1e-13)
    assert np.allclose(oracle.forces_xm(x, m, eps2, 3.0 * G), 3.0 * F, rtol=1e-13)
    mirror = x * np.array([-1.0, 1.0, 1.0])
    assert np.allclose(oracle.forces_xm(mirror, m, eps2, G), F * np.array([-1.0, 1.0, 1.0]), rtol=1e-12)
    # linearity in the source masses
    m2 = RNG.random(n)
    assert np.allclose(oracle.forces_xm(x, m + m2, eps2, G),
                       F + oracle.forces_xm(x, m2, eps2, G), rtol=1e-11, atol=1e-12)


# ----------------------------------------------------------------------------- P6
def test_far_field_monopole():
    n, s, R = 3000, 0.01, 10.0
    cl = s * (RNG.random((n, 3)) - 0.5)
    m = RNG.random(n)
    com = (m[:, None] * cl).sum(0) / m.sum()
    probe = com + np.array([R, 0, 0])
    x = np.concatenate([cl, probe[None]], axis=0)
    mm = np.concatenate([m, [0.0]])
    F = oracle.forces_xm(x, mm, 1e-8, 1.0, targets=np.array([n]))[0]
    assert F[0] == pytest.approx(-m.sum() / R ** 2, rel=5 * (s / R) ** 2)
    assert abs(F[1]) + abs(F[2]) < 5 * (s / R) ** 2 * m.sum() / R ** 2


# ----------------------------------------------------------------------------- P7
EDS = Cosmology(H0=2.5, Om_M=1.0)
LCDM = Cosmology(H0=70.0, Om_M=0.3, Om_L=0.7)


def test_hubble_each_term():
    c = Cosmology(H0=3.0, Om_R=0.1, Om_M=0.2, Om_K=0.3, Om_L=0.4)
    a = 0.5
    assert oracle.hubble(c, a) == pytest.approx(3.0 * math.sqrt(0.1 * 16 + 0.2 * 8 + 0.3 * 4 + 0.4), rel=1e-15)
    assert oracle.hubble(c, 1.0) == pytest.approx(3.0, rel=1e-15)
    for name, expo in (("Om_R", -2.0), ("Om_M", -1.5), ("Om_K", -1.0), ("Om_L", 0.0)):
        single = Cosmology(H0=1.0, **{name: 1.0})
        assert oracle.hubble(single, 0.3) == pytest.approx(0.3 ** expo, rel=1e-14)


def test_eds_closed_form():
    """a = (1.5 H0 t)^{2/3}, H = 2/(3t)."""
    H0 = EDS.H0
    t = lambda a: (2.0 / (3.0 * H0)) * a ** 1.5
    assert oracle.time_of_a(EDS, 0.02) == pytest.approx(t(0.02), rel=1e-10)
    assert oracle.time_of_a(EDS, 1.0) == pytest.approx(t(1.0), rel=1e-10)
    a0, dt = 0.02, 0.013
    a1 = oracle.a_advance(EDS, a0, dt, 8192)
    assert a1 == pytest.approx((1.5 * H0 * (t(a0) + dt)) ** (2.0 / 3.0), rel=1e-10)
    assert oracle.hubble(EDS, a1) == pytest.approx(2.0 / (3.0 * (t(a0) + dt)), rel=1e-10)


def test_flat_lcdm_closed_form():
    """H0 t = (2 / (3 sqrt(Om_L))) asinh( sqrt(Om_L/Om_M) a^{3/2} );  H0 t0 = 0.9640993816 for (0.3, 0.7)."""
    f = lambda a: (2.0 / (3.0 * math.sqrt(0.7))) * math.asinh(math.sqrt(0.7 / 0.3) * a ** 1.5) / 70.0
    assert 70.0 * oracle.time_of_a(LCDM, 1.0) == pytest.approx(0.9640993816, rel=2e-10)
    assert oracle.time_of_a(LCDM, 1.0 / 51.0) == pytest.approx(f(1.0 / 51.0), rel=1e-10)
    # advance from z=50 to z=0 in 1000 steps of tau, as config 2 does
    tau = (f(1.0) - f(1.0 / 51.0)) / 1000.0
    a = 1.0 / 51.0
    for _ in range(1000):
        a = oracle.a_advance(LCDM, a, tau, 16)
    assert a == pytest.approx(1.0, rel=1e-9)
    # inverse closed form at an intermediate time
    tmid = f(1.0 / 51.0) + 400 * tau
    a_mid = (math.sqrt(0.3 / 0.7) * math.sinh(1.5 * math.sqrt(0.7) * 70.0 * tmid)) ** (2.0 / 3.0)
    assert oracle.a_advance(LCDM, 1.0 / 51.0, 400 * tau, 4000) == pytest.approx(a_mid, rel=1e-10)


def test_radiation_milne_desitter_closed_forms():
    rad = Cosmology(H0=1.7, Om_R=1.0)                                   # a = sqrt(2 H0 t)
    assert oracle.time_of_a(rad, 0.4) == pytest.approx(0.4 ** 2 / (2 * 1.7), rel=1e-10)
    t0 = 0.1 ** 2 / (2 * 1.7)
    assert oracle.a_advance(rad, 0.1, 0.05, 8192) == pytest.approx(math.sqrt(2 * 1.7 * (t0 + 0.05)), rel=1e-10)
    milne = Cosmology(H0=0.9, Om_K=1.0)                                 # a = H0 t
    assert oracle.time_of_a(milne, 0.6) == pytest.approx(0.6 / 0.9, rel=1e-10)
    assert oracle.a_advance(milne, 0.2, 0.3, 64) == pytest.approx(0.2 + 0.9 * 0.3, rel=1e-12)
    ds = Cosmology(H0=1.1, Om_L=1.0)                                    # a ~ exp(H0 t)
    assert oracle.a_advance(ds, 0.5, 0.7, 64) == pytest.approx(0.5 * math.exp(1.1 * 0.7), rel=1e-9)


def test_matter_radiation_and_open_closed_forms():
    Om_M, Om_R, H0 = 0.9, 0.1, 2.0
    mr = Cosmology(H0=H0, Om_R=Om_R, Om_M=Om_M)
    f = lambda a: (2.0 / (3.0 * Om_M ** 2)) * ((Om_M * a - 2 * Om_R) * math.sqrt(Om_M * a + Om_R)
                                               + 2 * Om_R ** 1.5) / H0
    for a in (0.05, 0.5, 1.0):
        assert oracle.time_of_a(mr, a) == pytest.approx(f(a), rel=1e-9)
    a1 = oracle.a_advance(mr, 0.05, f(0.5) - f(0.05), 4000)
    assert a1 == pytest.approx(0.5, rel=1e-9)
    Om_M, Om_K = 0.3, 0.7                                               # open: cycloid-like parametric form
    op = Cosmology(H0=H0, Om_M=Om_M, Om_K=Om_K)
    for eta in (0.5, 1.5, 2.5):
        a = (Om_M / (2 * Om_K)) * (math.cosh(eta) - 1.0)
        t = (Om_M / (2 * Om_K ** 1.5)) * (math.sinh(eta) - eta) / H0
        assert oracle.time_of_a(op, a) == pytest.approx(t, rel=1e-9)


def test_int_dt_over_a_pow_eds():
    """EdS: a = (t/t1)^{2/3} with t1 = 2/(3 H0): int dt/a^p has a closed form."""
    H0 = EDS.H0
    t1 = 2.0 / (3.0 * H0)
    a0, dt = 0.1, 0.02
    ta = t1 * a0 ** 1.5
    for p in (1.0, 2.0):
        q = 1.0 - 2.0 * p / 3.0
        want = t1 ** (2 * p / 3) * ((ta + dt) ** q - ta ** q) / q
        assert oracle.int_dt_over_a_pow(EDS, a0, dt, p, 2048) == pytest.approx(want, rel=1e-9)


def test_midstep_schedule():
    mids, ends = oracle.midstep_schedule(EDS, 0.02, 1e-3, 10)
    t1 = 2.0 / (3.0 * EDS.H0)
    t0 = t1 * 0.02 ** 1.5
    for i, (a, H) in enumerate(mids):
        tm = t0 + (i + 0.5) * 1e-3
        assert a == pytest.approx((tm / t1) ** (2 / 3), rel=1e-9)
        assert H == pytest.approx(2.0 / (3.0 * tm), rel=1e-9)
    assert ends[-1] == pytest.approx(((t0 + 10e-3) / t1) ** (2 / 3), rel=1e-9)
    mids, ends = oracle.midstep_schedule(None, 1.0, 1e-3, 3)
    assert mids == [(1.0, 0.0)] * 3 and ends == [1.0] * 4


# ----------------------------------------------------------------------------- P8
def _pm(x, m):
    return np.concatenate([np.asarray(x, dtype=np.float64), np.asarray(m, dtype=np.float64)[:, None]], axis=1)


def _two_body_circular(eps2, G=1.0, m1=1.0, m2=0.5, r=1.0):
    M = m1 + m2
    omega = math.sqrt(G * M / (r * r + eps2) ** 1.5)          # softened circular frequency
    x = np.array([[-m2 / M * r, 0, 0], [m1 / M * r, 0, 0]])
    v = np.array([[0, -m2 / M * r * omega, 0], [0, m1 / M * r * omega, 0]])
    return x, v, np.array([m1, m2]), omega


def _energy(st):
    d = st.diagnostics(1.0, with_potential=True)
    return d[7] + d[8]


def test_static_limit_is_leapfrog_circular_orbit():
    eps2 = 0.04
    x, v, m, omega = _two_body_circular(eps2)
    period = 2 * math.pi / omega
    errs = []
    for nsteps in (400, 800):
        st = oracle.State(_pm(x, m), np.concatenate([v, np.zeros((2, 1))], axis=1), eps2, 1.0)
        E0 = _energy(st)
        tau = period / nsteps
        worst = 0.0
        for _ in range(nsteps):
            st.step(tau, 1.0, 0.0)
            worst = max(worst, abs(_energy(st) - E0))
            assert np.linalg.norm(st.x[1] - st.x[0]) == pytest.approx(1.0, abs=2e-3)
        assert np.allclose(st.x, x, atol=5e-3)                # back to the start after one period
        assert np.allclose((st.m[:, None] * st.v).sum(0), 0.0, atol=1e-15)
        errs.append(np.linalg.norm(st.x - x))
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.05)   # second order: phase error ~ tau^2


def test_static_energy_error_second_order_and_time_reversal():
    n = 24
    x = RNG.random((n, 3))
    v = 0.3 * RNG.normal(size=(n, 3))
    m = RNG.random(n) / n
    pm = _pm(x, m)
    v4 = np.concatenate([v, np.zeros((n, 1))], axis=1)
    errs = []
    for tau, steps in ((2e-3, 100), (1e-3, 200)):
        st = oracle.State(pm, v4, 0.01, 1.0)
        E0 = _energy(st)
        for _ in range(steps):
            st.step(tau, 1.0, 0.0)
        errs.append(abs(_energy(st) - E0))
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.25)
    st = oracle.State(pm, v4, 0.01, 1.0)
    for _ in range(50):
        st.step(1e-3, 1.0, 0.0)
    st.v *= -1.0
    for _ in range(50):
        st.step(1e-3, 1.0, 0.0)
    assert np.allclose(st.x, x, atol=1e-13)
    assert np.allclose(-st.v, v, atol=1e-12)


# ----------------------------------------------------------------------------- P9
def test_one_step_worked_example(golden_dir):
    rows = _read_golden(os.path.join(golden_dir, "one_step_worked.txt"))
    pm = _pm([[0, 0, 0], [1, 2, 1]], [1.0, 125.0])
    vel = np.array([[0, 0, 0, 0], [0, 0, 8, 0]], dtype=np.float64)
    st = oracle.State(pm, vel, 16.0, 1.0)
    P0 = (st.m[:, None] * st.v).sum(0)
    st.step(0.25, 0.5, 4.0 / 3.0)
    for i, body in enumerate("AB"):
        want = [float(s) for s in rows[body]]
        assert np.allclose(st.x[i], want[:3], rtol=0, atol=1e-15)
        assert np.allclose(st.v[i], want[3:], rtol=0, atol=1e-15)
    assert np.allclose((st.m[:, None] * st.v).sum(0), 0.5 * P0, atol=1e-13)   # P' = cv P
    assert np.allclose(st.last_force(), [[1, 2, 2], [-1 / 125, -2 / 125, -2 / 125]], atol=1e-16)


def test_hubble_drag_without_forces():
    """G = 0: v^n = v^0 prod (1-H tau)/(1+H tau); continuous limit v ~ a^-2, second order in tau."""
    pm = _pm(RNG.random((5, 3)), np.ones(5))
    v0 = RNG.normal(size=(5, 4))
    v0[:, 3] = 0
    errs = []
    for steps in (50, 100):
        tau = 0.02 / steps
        mids, ends = oracle.midstep_schedule(EDS, 0.05, tau, steps)
        st = oracle.State(pm, v0, 0.01, 0.0)
        prod = 1.0
        for a, H in mids:
            st.step(tau, a, H)
            prod *= (1 - H * tau) / (1 + H * tau)
        assert np.allclose(st.v, v0[:, :3] * prod, rtol=1e-13)
        errs.append(abs(prod - (0.05 / ends[-1]) ** 2))
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.1)
    assert errs[1] < 1e-4


def test_momentum_law_with_forces():
    n = 50
    pm = _pm(RNG.random((n, 3)), RNG.random(n) / n)
    v0 = np.concatenate([0.2 * RNG.normal(size=(n, 3)), np.zeros((n, 1))], axis=1)
    st = oracle.State(pm, v0, 1e-3, 1.0)
    mids, _ = oracle.midstep_schedule(EDS, 0.1, 2e-3, 5)
    for a, H in mids:
        P = st.diagnostics(a)[1:4].copy()
        st.step(2e-3, a, H)
        cv = (1 - H * 2e-3) / (1 + H * 2e-3)
        assert np.allclose(st.diagnostics(a)[1:4], cv * P, rtol=1e-12, atol=1e-16)


# ----------------------------------------------------------------------------- diagnostics / P11
def test_diagnostics_definitions():
    n = 30
    x = RNG.random((n, 3))
    v = RNG.normal(size=(n, 3))
    m = RNG.random(n)
    st = oracle.State(_pm(x, m), np.concatenate([v, np.zeros((n, 1))], 1), 0.02, 1.5)
    a = 0.4
    d = st.diagnostics(a, with_potential=True)
    assert d[0] == pytest.approx(m.sum(), rel=1e-14)
    assert np.allclose(d[1:4], (m[:, None] * v).sum(0), rtol=1e-13)
    assert np.allclose(d[4:7], a * a * (m[:, None] * v).sum(0), rtol=1e-13)
    assert d[7] == pytest.approx(0.5 * a * a * (m * (v ** 2).sum(1)).sum(), rel=1e-13)
    dd = x[None] - x[:, None]
    s = np.sqrt((dd ** 2).sum(-1) + 0.02)
    pair = m[:, None] * m[None, :] / s
    np.fill_diagonal(pair, 0.0)
    assert d[8] == pytest.approx(-(1.5 / (2 * a)) * pair.sum(), rel=1e-13)
    assert np.allclose(d[9:12], (m[:, None] * x).sum(0) / m.sum(), rtol=1e-13)
    assert math.isnan(st.diagnostics(a)[8])


def test_layzer_irvine():
    """d(T+W)/dt = -H (2T + W) for eq. (1): time-integrated residual is O(tau^2)."""
    n = 64
    pm = _pm(RNG.random((n, 3)), np.full(n, 1.0 / n))
    v0 = np.zeros((n, 4))
    cosmo = Cosmology(H0=math.sqrt(8 * math.pi / 3), Om_M=1.0)
    res = []
    for steps in (40, 80):
        tau = 0.004 / steps
        mids, ends = oracle.midstep_schedule(cosmo, 0.05, tau, steps)
        st = oracle.State(pm, v0, 0.01 ** 2 * 25, 1.0)
        d = st.diagnostics(ends[0], True)
        E = [d[7] + d[8]]
        rhs = [oracle.hubble(cosmo, ends[0]) * (2 * d[7] + d[8])]
        for i, (a, H) in enumerate(mids):
            st.step(tau, a, H)
            d = st.diagnostics(ends[i + 1], True)
            E.append(d[7] + d[8])
            rhs.append(oracle.hubble(cosmo, ends[i + 1]) * (2 * d[7] + d[8]))
        rhs = np.array(rhs)
        integral = tau * (rhs.sum() - 0.5 * (rhs[0] + rhs[-1]))            # trapezoid
        res.append(abs(E[-1] - E[0] + integral))
        assert abs(E[-1] - E[0]) > 100 * res[-1]                            # non-vacuous: E changed a lot
    assert res[0] / res[1] == pytest.approx(4.0, rel=0.35)


# ----------------------------------------------------------------------------- P12: symplectic step, eq. (9)
def test_symplectic_force_free_closed_form():
    """G = 0 in EdS: w = a^2 v is constant and x moves by w * int dt/a^2, which has a closed form
    (a = (t/t1)^{2/3}: int dt/a^2 = -3 t1^{4/3} [t^{-1/3}])."""
    H0 = EDS.H0
    t1 = 2.0 / (3.0 * H0)
    a0, tau, steps = 0.05, 2e-3, 7
    t0 = t1 * a0 ** 1.5
    x0 = RNG.random((4, 3))
    w0 = RNG.normal(size=(4, 4))
    w0[:, 3] = 0
    st = oracle.State(_pm(x0, np.ones(4)), w0, 0.01, 0.0)
    a = a0
    for _ in range(steps):
        a = st.step_symplectic(EDS, a, tau)
    tf = t0 + steps * tau
    assert a == pytest.approx((tf / t1) ** (2 / 3), rel=1e-9)
    drift = -3.0 * t1 ** (4 / 3) * (tf ** (-1 / 3) - t0 ** (-1 / 3))
    assert np.allclose(st.v, w0[:, :3], rtol=0, atol=0)                    # cv = 1 exactly
    assert np.allclose(st.x, x0 + drift * w0[:, :3], rtol=1e-9)


def test_symplectic_conserves_canonical_momentum_exactly():
    """K adds ck * F with sum_k m_k F_k = 0 (P2) and cv = 1: sum m w is conserved to roundoff,
    unlike eqs. (3)-(5) where it decays by the drag factor (P9)."""
    n = 40
    pm = _pm(RNG.random((n, 3)), RNG.random(n) / n)
    w0 = np.concatenate([0.1 * RNG.normal(size=(n, 3)), np.zeros((n, 1))], axis=1)
    st = oracle.State(pm, w0, 1e-3, 1.0)
    P0 = (st.m[:, None] * st.v).sum(0)
    a = 0.1
    for _ in range(5):
        a = st.step_symplectic(LCDM, a, 1e-4)
    scale = (st.m[:, None] * np.abs(st.v)).sum()
    assert np.abs((st.m[:, None] * st.v).sum(0) - P0).max() <= 1e-13 * scale
    assert np.abs(st.v - w0[:, :3]).max() > 1e-3                            # non-vacuous: kicks happened


def test_symplectic_static_limit_is_leapfrog():
    """H0 -> 0 (a = 1): the integrals are tau/2, tau, tau/2 and eq. (9) is the plain D-K-D leapfrog."""
    static = Cosmology(H0=1e-30, Om_L=1.0)
    x, v, m, _ = _two_body_circular(0.04)
    s1 = oracle.State(_pm(x, m), np.concatenate([v, np.zeros((2, 1))], 1), 0.04, 1.0)
    s2 = oracle.State(_pm(x, m), np.concatenate([v, np.zeros((2, 1))], 1), 0.04, 1.0)
    for _ in range(20):
        s1.step_symplectic(static, 1.0, 0.01)
        s2.step(0.01, 1.0, 0.0)
    assert np.allclose(s1.x, s2.x, rtol=0, atol=1e-13) and np.allclose(s1.v, s2.v, rtol=0, atol=1e-13)


def test_symplectic_and_eqs_3_5_converge_to_each_other():
    """Both schemes integrate d(a^2 v)/dt = F/a: with v = w/a^2 their end states differ by O(tau^2)."""
    n = 24
    pm = _pm(RNG.random((n, 3)), np.full(n, 1.0 / n))
    v0 = np.concatenate([0.3 * RNG.normal(size=(n, 3)), np.zeros((n, 1))], axis=1)
    a0, T = 0.2, 0.02
    diffs = []
    for steps in (40, 80):
        tau = T / steps
        s1 = oracle.State(pm, v0, 0.05 ** 2, 1.0)
        mids, ends = oracle.midstep_schedule(EDS, a0, tau, steps)
        for a, H in mids:
            s1.step(tau, a, H)
        w0 = v0.copy()
        w0[:, :3] *= a0 * a0
        s2 = oracle.State(pm, w0, 0.05 ** 2, 1.0)
        a = a0
        for _ in range(steps):
            a = s2.step_symplectic(EDS, a, tau)
        assert a == pytest.approx(ends[-1], rel=1e-9)
        diffs.append(np.abs(s1.x - s2.x).max() + np.abs(s1.v - s2.v / a ** 2).max())
        assert np.abs(s1.x - pm[:, :3]).max() > 100 * diffs[-1]            # non-vacuous
    assert diffs[0] / diffs[1] == pytest.approx(4.0, rel=0.25)


# ----------------------------------------------------------------------------- P13: eq. (10) and background
def test_deformation_source_is_a_fixed_extra_body():
    """Eq. (10): the term 'acts like a mass particle located in a fixed position': it must
    equal what eq. (1) gives when a body of mass S/G is appended at x_psi; and the two-body closed form."""
    n, G, eps2, S = 17, 2.5, 0.03 ** 2, 0.7
    x = RNG.random((n, 3))
    m = RNG.random(n)
    xpsi = np.array([0.3, -0.2, 1.1])
    base = oracle.forces_xm(x, m, eps2, G)
    got = oracle.add_external(x, base.copy(), eps2, G, deformation=(xpsi, S))
    want = oracle.forces_xm(np.vstack([x, xpsi]), np.append(m, S / G), eps2, G)[:n]
    assert np.allclose(got, want, rtol=1e-13, atol=1e-15)
    d = xpsi - x[3]
    r2 = d @ d
    assert np.allclose(got[3] - base[3], S * d / (r2 + eps2) ** 1.5, rtol=1e-14)      # toward x_psi
    sub = oracle.add_external(x, base[[5, 2]].copy(), eps2, G, targets=[5, 2], deformation=(xpsi, S))
    assert np.allclose(sub, want[[5, 2]], rtol=1e-13)


def test_background_term_closed_form_and_sphere_cancellation():
    """F += (4 pi/3) G rho (x - c): linear closed form; and it cancels the pull of a homogeneous sphere
    (shell theorem: -G M(<r)/r^2 = -(4 pi/3) G rho r) up to the discreteness of the lattice."""
    G, rho = 1.7, 3.0
    x = RNG.random((5, 3))
    c = np.array([0.5, 0.4, 0.6])
    got = oracle.add_external(x, np.zeros((5, 3)), 0.01, G, background=(c, rho))
    assert np.allclose(got, (4 * math.pi / 3) * G * rho * (x - c), rtol=1e-15)
    side = 28
    g = (np.arange(side) + 0.5) / side - 0.5
    X = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    X = X[(X ** 2).sum(1) <= 0.25]                                   # lattice points inside R = 0.5
    m = np.full(len(X), 1.0 / side ** 3)                             # density 1
    probes = np.array([[0.2, 0.1, -0.1], [-0.3, 0.05, 0.2], [0.0, 0.25, 0.0]])
    pts = np.vstack([X, probes])
    mm = np.append(m, np.zeros(3))                                   # massless probes
    tg = np.arange(len(X), len(X) + 3)
    grav = oracle.forces_xm(pts, mm, (0.5 / side) ** 2, G, tg)
    tot = oracle.add_external(pts, grav.copy(), 0.0, G, targets=tg, background=(np.zeros(3), 1.0))
    assert np.all(np.linalg.norm(tot, axis=1) <= 0.03 * np.linalg.norm(grav, axis=1))


def test_step_with_external_terms_matches_composition():
    """State.step with the external terms = drift, (eq. 1 + external), kick, drift written out here."""
    n = 12
    x0 = RNG.random((n, 3))
    m = RNG.random(n) / n
    v0 = 0.1 * RNG.normal(size=(n, 3))
    st = oracle.State(_pm(x0, m), np.concatenate([v0, np.zeros((n, 1))], 1), 1e-3, 1.0)
    st.deformation = (np.array([0.5, 0.5, 2.0]), 0.3)
    st.background = (np.array([0.5, 0.5, 0.5]), 0.8)
    tau, a, H = 1e-2, 0.5, 0.7
    st.step(tau, a, H)
    xh = x0 + 0.5 * tau * v0
    F = oracle.forces_xm(xh, m, 1e-3, 1.0)
    F = F + 0.3 * (st.deformation[0] - xh) / (((st.deformation[0] - xh) ** 2).sum(1, keepdims=True) + 1e-3) ** 1.5
    F = F + (4 * math.pi / 3) * 0.8 * (xh - 0.5)
    v1 = v0 * (1 - H * tau) / (1 + H * tau) + F * tau / (a ** 3 * (1 + H * tau))
    assert np.allclose(st.v, v1, rtol=1e-12, atol=1e-15)
    assert np.allclose(st.x, xh + 0.5 * tau * v1, rtol=1e-13)


# ----------------------------------------------------------------------------- P14: headless snapshot (f4)
def _splat_rational(pos, axis, window, width, height):
    """Brute force in exact rational arithmetic: valid when every input is dyadic and the scale
    width/(u1-u0) is a power of two, so that the FP32 pixel decision of reading G23 is exact."""
    iu, iv = (axis + 1) % 3, (axis + 2) % 3
    u0, u1, v0, v1 = [Fraction(float(c)) for c in window[:4]]
    w0, w1 = float(window[4]), float(window[5])                     # may be -inf / +inf (no slab)
    img = [[0] * width for _ in range(height)]
    for p in pos:
        u, v, w = Fraction(float(p[iu])), Fraction(float(p[iv])), Fraction(float(p[axis]))
        if not (w0 <= w < w1):
            continue
        tu, tv = (u - u0) * width / (u1 - u0), (v - v0) * height / (v1 - v0)
        if 0 <= tu < width and 0 <= tv < height:
            img[math.floor(tv)][math.floor(tu)] += 1
    return np.array(img, dtype=np.uint32)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_splat_brute_force_exact_on_dyadic_inputs(axis):
    """Pixel = floor((u - u0) W / (u1 - u0)); image axes (u, v) cyclic after `axis`; slab on the depth."""
    n = 3000
    pos = (RNG.integers(-256, 1280, size=(n, 3)) / 1024.0).astype(np.float32)   # dyadic, some outside [0,1)
    pm = np.concatenate([pos, np.ones((n, 1), np.float32)], 1)
    for window, (W, H) in ((((0.0, 1.0, 0.0, 1.0, 0.25, 0.75)), (32, 16)),
                           ((-0.25, 0.75, 0.5, 1.0, -np.inf, np.inf), (64, 8)),
                           ((0.5, 0.625, 0.0, 0.25, 0.0, 1.0), (4, 4))):
        got = oracle.splat(pm, axis, window, W, H)
        want = _splat_rational(pos, axis, window, W, H)
        assert got.dtype == np.uint32 and got.shape == (H, W)
        assert np.array_equal(got, want)
        assert want.sum() > 0


def test_splat_total_and_marginals_match_numpy_histogram():
    """Sum of the image = particles inside window and slab; its marginals = numpy.histogram of u and v
    (inputs dyadic with a power-of-two bin width, so numpy's FP64 binning is exact as well)."""
    n = 20000
    pos = (RNG.integers(0, 4096, size=(n, 3)) / 4096.0).astype(np.float32)
    pm = np.concatenate([pos, np.zeros((n, 1), np.float32)], 1)
    img = oracle.splat(pm, 2, (0.0, 1.0, 0.0, 1.0, 0.125, 0.5), 64, 32)
    sel = (pos[:, 2] >= 0.125) & (pos[:, 2] < 0.5)
    assert img.sum() == sel.sum()
    hu, _ = np.histogram(pos[sel, 0].astype(np.float64), bins=64, range=(0.0, 1.0))
    hv, _ = np.histogram(pos[sel, 1].astype(np.float64), bins=32, range=(0.0, 1.0))
    assert np.array_equal(img.sum(0), hu) and np.array_equal(img.sum(1), hv)
    # the upper edges are exclusive: a particle exactly at u1 is not counted (numpy's last bin is closed)
    edge = np.array([[1.0, 0.5, 0.25, 1.0], [0.5, 1.0, 0.25, 1.0], [0.5, 0.5, 0.5, 1.0], [0.0, 0.0, 0.125, 1.0]],
                    dtype=np.float32)
    e = oracle.splat(edge, 2, (0.0, 1.0, 0.0, 1.0, 0.125, 0.5), 4, 4)
    assert e.sum() == 1 and e[0, 0] == 1


def test_splat_pixel_decision_is_fp32():
    """Reading G23: the pixel is decided in FP32, (u - u0) * (W / (u1 - u0)) with each op rounded once.
    Independent restatement with numpy float32 scalars on non-dyadic inputs."""
    n = 5000
    pos = RNG.random((n, 3)).astype(np.float32)
    pm = np.concatenate([pos, np.ones((n, 1), np.float32)], 1)
    win = np.array([0.1, 0.9, 0.2, 0.7, 0.0, 1.0], dtype=np.float32)
    W, H = 37, 23
    su = np.float32(W) / (win[1] - win[0])
    sv = np.float32(H) / (win[3] - win[2])
    tu = (pos[:, 1] - win[0]) * su          # axis 0: u = y, v = z
    tv = (pos[:, 2] - win[2]) * sv
    assert tu.dtype == np.float32
    ok = (tu >= 0) & (tu < W) & (tv >= 0) & (tv < H)
    want = np.zeros((H, W), dtype=np.uint32)
    np.add.at(want, (np.floor(tv[ok]).astype(int), np.floor(tu[ok]).astype(int)), 1)
    assert np.array_equal(oracle.splat(pm, 0, win, W, H), want)


# ----------------------------------------------------------------------------- P15: tracer power spectrum (f3)
def _series(v):
    """[S, k, 3] -> ring rows [S, k, 4] float32."""
    S, k, _ = v.shape
    out = np.zeros((S, k, 4), dtype=np.float32)
    out[:, :, :3] = v
    out[:, :, 3] = 7.0          # the tag column must be ignored
    return out


def test_spectrum_sinusoid_and_constant_closed_forms():
    """v_x[s] = A cos(2 pi f0 s / S + phi): P[f0] = S A^2 / 4 (0 < f0 < S/2), 0 elsewhere;
    a constant c in v_y: P[0] = S c^2; Nyquist (-1)^s B in v_z: P[S/2] = S B^2."""
    S, f0, A, phi, c, B = 64, 5, 0.75, 0.3, 0.5, 0.25
    s = np.arange(S)
    v = np.zeros((S, 2, 3))
    v[:, 0, 0] = A * np.cos(2 * np.pi * f0 * s / S + phi)
    v[:, 1, 1] = c
    v[:, 1, 2] = B * (-1.0) ** s
    ser = _series(v)
    P = oracle.trace_spectrum(ser)
    assert P.shape == (2, S // 2 + 1)
    x32 = ser[:, 0, 0].astype(np.float64)                           # the float32-rounded series
    want0 = np.zeros(S // 2 + 1)
    want0[f0] = S * A * A / 4
    assert np.allclose(P[0], want0, atol=2e-6 * S * A * A)          # float32 rounding of the samples
    want1 = np.zeros(S // 2 + 1)
    want1[0], want1[S // 2] = S * c * c, S * B * B
    assert np.allclose(P[1], want1, atol=1e-12)                     # 0.5, +-0.25 are exact in float32
    assert abs(P[0].sum() * 2 - (x32 ** 2).sum()) < 1e-5            # only interior bins are occupied


@pytest.mark.parametrize("S", [16, 45, 100])
def test_spectrum_parseval_and_numpy_rfft(S):
    """Full-circle sum of P = sum_s |v[s]|^2 (one-sided bins doubled except 0 and Nyquist), and
    P = sum_c |rfft(v_c)|^2 / S (special case: the definition is a DFT)."""
    k = 5
    ser = _series(RNG.normal(size=(S, k, 3)))
    P = oracle.trace_spectrum(ser)
    v = ser[:, :, :3].astype(np.float64)
    wgt = np.full(S // 2 + 1, 2.0)
    wgt[0] = 1.0
    if S % 2 == 0:
        wgt[-1] = 1.0
    assert np.allclose((P * wgt).sum(1), (v ** 2).sum((0, 2)), rtol=1e-12)
    F = np.fft.rfft(v, axis=0)                                      # [S//2+1, k, 3]
    assert np.allclose(P, (np.abs(F) ** 2).sum(2).T / S, rtol=1e-10, atol=1e-12)


def test_spectrum_time_shift_invariance_and_component_sum():
    """A cyclic shift of the record changes only phases; components add."""
    S, k = 40, 3
    v = RNG.normal(size=(S, k, 3))
    P = oracle.trace_spectrum(_series(v))
    assert np.allclose(oracle.trace_spectrum(_series(np.roll(v, 7, axis=0))), P, rtol=1e-9, atol=1e-12)
    parts = 0
    for c in range(3):
        vc = np.zeros_like(v)
        vc[:, :, c] = v[:, :, c]
        parts = parts + oracle.trace_spectrum(_series(vc))
    assert np.allclose(parts, P, rtol=1e-12, atol=1e-14)


# ----------------------------------------------------------------------------- P16: cold homogeneous sphere
def test_cold_lattice_sphere_follows_the_shell_ode():
    """Force and step together, at N ~ 2000, against one scalar equation.  A cold homogeneous sphere (lattice
    points inside R, equal masses, mean density rho) contracts self-similarly: by the shell theorem the force on
    a shell that started at r0 and now sits at s r0 is -(4 pi/3) G rho r0 / s^2 (mass inside is conserved), so
    every shell obeys the SAME scalar recurrence when eqs. (3)-(5) are applied to s:
        s += tau/2 u;  u = u (1-H tau)/(1+H tau) - K / s^2 * tau / (a^3 (1+H tau));  s += tau/2 u,
    K = (4 pi/3) G rho.  (Config-2 units: this is the global contraction of reading G7 -- 19 % in 10 steps.)"""
    side, G, rho = 16, 3 * 0.3 * 70.0 ** 2 / (8 * math.pi), 1.0
    cosmo = Cosmology(H0=70.0, Om_M=0.3, Om_L=0.7)
    tau, a0, steps = 1.37251071e-5, 1.0 / 51.0, 30
    g = (np.arange(side) + 0.5) / side - 0.5
    X = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    X = X[np.linalg.norm(X, axis=1) < 0.5]
    n = len(X)
    pm = _pm(X, np.full(n, rho / side ** 3))
    st = oracle.State(pm, np.zeros((n, 4), np.float32), (0.05 / side) ** 2, G)
    mids, _ = oracle.midstep_schedule(cosmo, a0, tau, steps)
    K = 4 * math.pi / 3 * G * rho
    s, u = 1.0, 0.0
    r0 = np.linalg.norm(X, axis=1)
    inner = (r0 > 0.1) & (r0 < 0.4)               # away from the centre's lattice noise and the ragged surface
    for k, (a, H) in enumerate(mids):
        st.step(tau, a, H)
        s += 0.5 * tau * u
        u = u * (1 - H * tau) / (1 + H * tau) - K / s ** 2 * tau / (a ** 3 * (1 + H * tau))
        s += 0.5 * tau * u
        if k + 1 in (10, 20, 30):
            q = np.linalg.norm(st.x, axis=1)[inner] / r0[inner]
            assert abs(np.median(q) - s) < 0.01 * s, (k + 1, np.median(q), s)
            assert np.percentile(q, 90) - np.percentile(q, 10) < 0.06 * s          # self-similar
    assert 0.35 < s < 0.45                        # 30 steps: the sphere has shrunk to ~41 %
