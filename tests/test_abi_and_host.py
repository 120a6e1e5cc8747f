"""CPU-side checks (-m "not gpu"): libcolatus loads and exports every symbol include/colatus.h
declares; the host-only FP64 Friedmann helpers (eq. 2) match closed forms; argument checks that
need no device."""
import math
import os
import re

import pytest

from paper_1208_3444_b200 import binding as B
from paper_1208_3444_b200 import build as cuda_build
from paper_1208_3444_b200.inputs import Cosmology

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    cuda_build.build()


def test_every_declared_symbol_is_exported_and_bound():
    header = open(os.path.join(ROOT, "include", "colatus.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(colatus_[a-z_0-9]+)\s*\(", header))
    assert len(declared) >= 25
    handle = B.lib()
    for name in declared:
        assert hasattr(handle, name), f"{name} not exported by libcolatus.so"
    assert declared == set(B.SIGNATURES), declared ^ set(B.SIGNATURES)


def test_probe_library_is_separate_and_exports_its_header():
    """Microbenchmarks live in libcolatus_probe.so (include/colatus_probe.h), not in the product ABI."""
    from paper_1208_3444_b200 import probe as P
    header = open(os.path.join(ROOT, "include", "colatus_probe.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(colatus_probe_[a-z_0-9]+)\s*\(", header))
    assert declared == set(P.SIGNATURES) and len(declared) == 2
    handle = P.lib()
    for name in declared:
        assert hasattr(handle, name)
    import subprocess
    product = subprocess.check_output(["nm", "-D", "--defined-only", B.LIB_PATH], text=True)
    assert "probe" not in product and "calibrate" not in product
    assert P.lib().colatus_probe_pipe(0, 99, None) == -1           # argument check needs no device


def test_library_does_not_link_torch_or_oracle():
    import subprocess
    out = subprocess.check_output(["ldd", B.LIB_PATH], text=True)
    assert "torch" not in out and "oracle" not in out


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1208_3444_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert not re.search(r"#\s*include[^\n]*oracle", text) and "liboracle" not in text, f


def test_workspace_bytes_is_host_arithmetic():
    assert B.colatus_workspace_bytes(0) == 0
    assert B.colatus_workspace_bytes(-5) == 0
    # below 20480 bodies: staged copy + 64 split partials + scratch: ~1.1 KB per body
    w4k = B.colatus_workspace_bytes(4096)
    assert w4k % 256 == 0 and 64 * 16 * 4096 < w4k < 8 * (1 << 20)
    # symmetric kernel (colatus_force_plan): all partial rows while they fit 512 MiB ((24 + 31) rows of 64 x 4096
    # bodies at 262144) ...
    w18 = B.colatus_workspace_bytes(1 << 18)
    rows18 = (24 + 31) * 64 * 4096 * 16
    assert w18 % 256 == 0 and rows18 < w18 < rows18 + 30 * (1 << 20)
    # ... beyond that 32 rows per launch, the evaluation chunked over block distances (measured knee,
    # profiles/r03_workspace_rows_sweep.md): VERDICT r2 bounds 0.6 GiB at 2^20, 2.5 GiB at 2^22
    w20, w22 = B.colatus_workspace_bytes(1 << 20), B.colatus_workspace_bytes(1 << 22)
    assert w20 % 256 == 0 and (512 << 20) < w20 <= int(0.6 * (1 << 30))
    assert (2 << 30) < w22 <= int(2.5 * (1 << 30))
    # non-decreasing in n: a workspace sized for n_max serves every n <= n_max
    sizes = [B.colatus_workspace_bytes(n) for n in (1, 100, 4096, 20479, 20480, 24576, 32768, 65535, 65536, 131071, 131072, 200000, 262144, 400000, 524288, 1 << 20, 1500000, 1 << 22)]
    assert all(a <= b for a, b in zip(sizes, sizes[1:]))


def test_uninitialised_calls_fail_loudly_without_a_device():
    assert B.lib().colatus_forces(None, 1, 0.1, None, None) == B.NOT_INITIALISED
    assert "colatus_init" in B.colatus_last_error()
    assert B.lib().colatus_step(1e-3, 1.0, 0.0) == B.NOT_INITIALISED
    with pytest.raises(B.ColatusError):
        B.colatus_diagnostics(1.0)


def test_static_entry_point_limit_and_argument_checks_need_no_device():
    """colatus_forces_static (the entry point for callers who cannot allocate a workspace): the binding's limit is
    the header's, and the argument checks come before any CUDA call."""
    header = open(os.path.join(ROOT, "include", "colatus.h")).read()
    assert int(re.search(r"#define\s+COLATUS_STATIC_MAX_N\s+(\d+)", header).group(1)) == B.STATIC_MAX_N
    assert B.lib().colatus_forces_static(None, 10, 1e-4, 1.0, None, None) == B.INVALID_ARG
    assert B.lib().colatus_forces_static(16, B.STATIC_MAX_N + 1, 1e-4, 1.0, 32, None) == B.INVALID_ARG
    assert "COLATUS_STATIC_MAX_N" in B.colatus_last_error()


def test_step_coefficients_worked_example():
    """tests/golden/one_step_worked.txt: tau=1/4, a=1/2, H=4/3 -> cv = 1/2, ck = 3/2."""
    d1, cv, ck, d2 = B.colatus_step_coefficients(0.25, 0.5, 4.0 / 3.0)
    assert (d1, d2) == (0.125, 0.125)
    assert cv == pytest.approx(0.5, rel=1e-15) and ck == pytest.approx(1.5, rel=1e-15)
    with pytest.raises(B.ColatusError):
        B.colatus_step_coefficients(1.0, 1.0, -1.0)
    with pytest.raises(B.ColatusError):
        B.colatus_step_coefficients(1.0, 0.0, 0.0)


# ---- eq. (2) host helpers against closed forms ------------------------------------
def test_hubble():
    c = Cosmology(H0=3.0, Om_R=0.1, Om_M=0.2, Om_K=0.3, Om_L=0.4)
    assert B.colatus_hubble(c, 0.5) == pytest.approx(3.0 * math.sqrt(1.6 + 1.6 + 1.2 + 0.4), rel=1e-15)
    assert math.isnan(B.colatus_hubble(c, 0.0))


def test_eds():
    c = Cosmology(H0=2.894405, Om_M=1.0)
    t = lambda a: (2.0 / (3.0 * c.H0)) * a ** 1.5
    assert B.colatus_time_of_a(c, 0.02) == pytest.approx(t(0.02), rel=1e-12)
    assert B.colatus_a_advance(c, 0.02, 0.013) == pytest.approx((1.5 * c.H0 * (t(0.02) + 0.013)) ** (2 / 3), rel=1e-11)
    assert B.colatus_a_advance(c, 0.5, -0.01) == pytest.approx((1.5 * c.H0 * (t(0.5) - 0.01)) ** (2 / 3), rel=1e-11)
    t1 = 2.0 / (3.0 * c.H0)
    ta = t1 * 0.1 ** 1.5
    for p in (1.0, 2.0):
        q = 1.0 - 2.0 * p / 3.0
        want = t1 ** (2 * p / 3) * ((ta + 0.02) ** q - ta ** q) / q
        assert B.colatus_int_dt_over_a_pow(c, 0.1, 0.02, p) == pytest.approx(want, rel=1e-10)


def test_symplectic_coefficients_eds_closed_form():
    """Eq. (9) integrals in EdS, a = (t/t1)^{2/3}: int dt/a^p = t1^{2p/3} [t^q]/q, q = 1 - 2p/3."""
    c = Cosmology(H0=2.894405, Om_M=1.0)
    t1 = 2.0 / (3.0 * c.H0)
    a0, tau = 0.1, 0.02
    ta = t1 * a0 ** 1.5

    def integral(p, t_from, t_to):
        q = 1.0 - 2.0 * p / 3.0
        return t1 ** (2 * p / 3) * (t_to ** q - t_from ** q) / q

    d1, cv, ck, d2, a_end = B.colatus_symplectic_coefficients(c, a0, tau)
    assert cv == 1.0
    assert d1 == pytest.approx(integral(2.0, ta, ta + 0.5 * tau), rel=1e-10)
    assert d2 == pytest.approx(integral(2.0, ta + 0.5 * tau, ta + tau), rel=1e-10)
    assert ck == pytest.approx(integral(1.0, ta, ta + tau), rel=1e-10)
    assert a_end == pytest.approx(((ta + tau) / t1) ** (2 / 3), rel=1e-11)
    with pytest.raises(B.ColatusError):
        B.colatus_symplectic_coefficients(c, 0.0, tau)
    assert B.lib().colatus_set_deformation(None, 1.0) == B.NOT_INITIALISED
    assert B.lib().colatus_set_background(None, 1.0) == B.NOT_INITIALISED


def test_flat_lcdm():
    c = Cosmology(H0=70.0, Om_M=0.3, Om_L=0.7)
    f = lambda a: (2.0 / (3.0 * math.sqrt(0.7))) * math.asinh(math.sqrt(0.7 / 0.3) * a ** 1.5) / 70.0
    assert 70.0 * B.colatus_time_of_a(c, 1.0) == pytest.approx(0.9640993816, rel=2e-10)
    assert B.colatus_time_of_a(c, 1 / 51) == pytest.approx(f(1 / 51), rel=1e-12)
    assert B.colatus_a_advance(c, 1 / 51, f(1.0) - f(1 / 51)) == pytest.approx(1.0, rel=1e-11)


def test_other_closed_forms():
    rad = Cosmology(H0=1.7, Om_R=1.0)
    assert B.colatus_time_of_a(rad, 0.4) == pytest.approx(0.16 / 3.4, rel=1e-12)
    assert B.colatus_a_advance(rad, 0.1, 0.05) == pytest.approx(math.sqrt(2 * 1.7 * (0.01 / 3.4 + 0.05)), rel=1e-11)
    milne = Cosmology(H0=0.9, Om_K=1.0)
    assert B.colatus_time_of_a(milne, 0.6) == pytest.approx(0.6 / 0.9, rel=1e-12)
    assert B.colatus_a_advance(milne, 0.2, 0.3) == pytest.approx(0.47, rel=1e-12)
    ds = Cosmology(H0=1.1, Om_L=1.0)
    assert B.colatus_a_advance(ds, 0.5, 0.7) == pytest.approx(0.5 * math.exp(0.77), rel=1e-11)
    assert math.isinf(B.colatus_time_of_a(ds, 1.0))
    mr = Cosmology(H0=2.0, Om_R=0.1, Om_M=0.9)
    f = lambda a: (2.0 / (3.0 * 0.81)) * ((0.9 * a - 0.2) * math.sqrt(0.9 * a + 0.1) + 2 * 0.1 ** 1.5) / 2.0
    assert B.colatus_time_of_a(mr, 0.5) == pytest.approx(f(0.5), rel=1e-11)
    op = Cosmology(H0=2.0, Om_M=0.3, Om_K=0.7)
    eta = 1.5
    a = (0.3 / 1.4) * (math.cosh(eta) - 1.0)
    assert B.colatus_time_of_a(op, a) == pytest.approx((0.3 / (2 * 0.7 ** 1.5)) * (math.sinh(eta) - eta) / 2.0, rel=1e-11)


def test_library_and_oracle_schedules_agree():
    """The two independent Friedmann integrators give the same mid-step (a, H) for configs 1 and 2."""
    import oracle
    from paper_1208_3444_b200.inputs import CONFIGS
    for idx in (1, 2):
        cfg = CONFIGS[idx]
        mids, ends = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, 10)
        a = cfg.a_start
        for (am, Hm), ae in zip(mids, ends[1:]):
            a_mid = B.colatus_a_advance(cfg.cosmo, a, 0.5 * cfg.tau)
            assert a_mid == pytest.approx(am, rel=1e-9)
            assert B.colatus_hubble(cfg.cosmo, a_mid) == pytest.approx(Hm, rel=1e-9)
            a = B.colatus_a_advance(cfg.cosmo, a_mid, 0.5 * cfg.tau)
            assert a == pytest.approx(ae, rel=1e-9)


def test_config_constants():
    """Readings G13: the constants the configs leave open."""
    from paper_1208_3444_b200.inputs import CONFIGS
    c1, c2 = CONFIGS[1], CONFIGS[2]
    assert c1.cosmo.H0 == pytest.approx(2.894405, rel=1e-6)
    assert c2.G == pytest.approx(175.46832, rel=1e-7)
    t0 = B.colatus_time_of_a(c2.cosmo, 1.0)
    ti = B.colatus_time_of_a(c2.cosmo, 1.0 / 51.0)
    assert ti == pytest.approx(4.7741223e-5, rel=1e-6)
    assert (t0 - ti) / 1000.0 == pytest.approx(c2.tau, rel=1e-8)
