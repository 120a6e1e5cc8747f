"""CPU oracle for the COLATUS hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes wrapper over `colatus_oracle.c` (plain C, FP64, OpenMP over
targets).  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
`cpu_baseline` / `--impl reference` legs may import this package; the product
package `paper_1208_3444_b200` never does, and this package never imports it.

Inputs are the same float32 arrays handed to the GPU, promoted exactly to
double here.  See the header of `colatus_oracle.c` for citations and pins.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import c_double, c_int, c_int64, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "colatus_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                               "-ffp-contract=off", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(c_double)
        lib.oracle_num_threads.restype = c_int
        lib.oracle_forces.argtypes = [c_void_p, c_void_p, c_int64, c_double, c_double,
                                      c_void_p, c_int64, c_void_p, c_void_p]
        lib.oracle_forces.restype = None
        lib.oracle_step.argtypes = [c_void_p, c_void_p, c_void_p, c_int64, c_double, c_double,
                                    c_double, c_double, c_double, c_void_p]
        lib.oracle_step.restype = None
        lib.oracle_step_coeffs.argtypes = [c_void_p, c_void_p, c_void_p, c_int64, c_double, c_double,
                                           c_double, c_double, c_double, c_double, c_void_p]
        lib.oracle_step_coeffs.restype = None
        lib.oracle_add_external.argtypes = [c_void_p, c_void_p, c_int64, c_double, c_double, c_void_p,
                                            c_double, c_double, c_void_p, c_void_p]
        lib.oracle_add_external.restype = None
        lib.oracle_step_coeffs_ext.argtypes = [c_void_p, c_void_p, c_void_p, c_int64, c_double, c_double,
                                               c_double, c_double, c_double, c_double,
                                               c_double, c_void_p, c_double, c_void_p, c_void_p]
        lib.oracle_step_coeffs_ext.restype = None
        lib.oracle_hubble.argtypes = [c_double] * 6
        lib.oracle_hubble.restype = c_double
        lib.oracle_a_advance.argtypes = [c_double] * 7 + [c_int]
        lib.oracle_a_advance.restype = c_double
        lib.oracle_time_of_a.argtypes = [c_double] * 6 + [c_int64]
        lib.oracle_time_of_a.restype = c_double
        lib.oracle_int_dt_over_a_pow.argtypes = [c_double] * 8 + [c_int]
        lib.oracle_int_dt_over_a_pow.restype = c_double
        lib.oracle_diagnostics.argtypes = [c_void_p, c_void_p, c_void_p, c_int64, c_double, c_double,
                                           c_double, c_int, c_void_p]
        lib.oracle_diagnostics.restype = None
        lib.oracle_splat.argtypes = [c_void_p, c_int64, c_int, c_void_p, c_int, c_int, c_void_p]
        lib.oracle_splat.restype = None
        lib.oracle_trace_spectrum.argtypes = [c_void_p, c_int64, c_int64, c_void_p]
        lib.oracle_trace_spectrum.restype = None
        del dp
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _p(a: np.ndarray):
    return a.ctypes.data_as(c_void_p)


def _c64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def forces_xm(x, m, eps2, G, targets=None, potential=False):
    """Eq. (1) on double arrays x [n,3], m [n].  Returns acc [k,3] (and phi [k])."""
    x = _c64(x)
    m = _c64(m)
    n = x.shape[0]
    if targets is None:
        tptr, k = None, n
    else:
        targets = np.ascontiguousarray(targets, dtype=np.int64)
        tptr, k = _p(targets), targets.shape[0]
    acc = np.empty((k, 3), dtype=np.float64)
    phi = np.empty(k, dtype=np.float64) if potential else None
    _load().oracle_forces(_p(x), _p(m), n, float(eps2), float(G), tptr, k, _p(acc),
                          _p(phi) if potential else None)
    return (acc, phi) if potential else acc


def forces(pos_mass, eps2, G, targets=None, potential=False):
    """Eq. (1) on the float32 [n,4] body array the GPU receives (promoted exactly)."""
    pm = np.asarray(pos_mass)
    return forces_xm(pm[:, :3].astype(np.float64), pm[:, 3].astype(np.float64),
                     eps2, G, targets, potential)


def add_external(x, acc, eps2, G, targets=None, deformation=None, background=None):
    """Adds eq. (10) (deformation = (x_psi[3], S)) and / or the mean-density background term
    (background = (centre[3], rho_bar)) to acc [k,3] for the targets (in place; returns acc)."""
    x = _c64(x)
    xpsi, S = (np.zeros(3), 0.0) if deformation is None else (_c64(deformation[0]), float(deformation[1]))
    cen, rho = (np.zeros(3), 0.0) if background is None else (_c64(background[0]), float(background[1]))
    if targets is None:
        tptr, k = None, acc.shape[0]
    else:
        targets = np.ascontiguousarray(targets, dtype=np.int64)
        tptr, k = _p(targets), targets.shape[0]
    assert acc.dtype == np.float64 and acc.flags.c_contiguous and acc.shape == (k, 3)
    _load().oracle_add_external(_p(x), tptr, k, float(eps2), S, _p(xpsi), float(G), rho, _p(cen), _p(acc))
    return acc


def splat(pos_mass, axis, window, width, height):
    """Particle-count image of the positions (NEXT row f4; Fig. 1 PAPER.md:83-85;
    reading G23).  pos_mass: float32 [n,4]; window = (u0, u1, v0, v1, w0, w1).  uint32 [height, width]."""
    pm = np.ascontiguousarray(pos_mass, dtype=np.float32)
    assert pm.ndim == 2 and pm.shape[1] == 4
    win = np.ascontiguousarray(window, dtype=np.float32)
    assert win.shape == (6,)
    img = np.empty((int(height), int(width)), dtype=np.uint32)
    _load().oracle_splat(_p(pm), pm.shape[0], int(axis), _p(win), int(width), int(height), _p(img))
    return img


def trace_spectrum(series):
    """Periodogram of the tracer velocity series (NEXT row f3; reading G24).
    series: float32 [S, k, 4] rows of the tracer ring.  float64 [k, S//2 + 1]."""
    sr = np.ascontiguousarray(series, dtype=np.float32)
    assert sr.ndim == 3 and sr.shape[2] == 4
    S, k = sr.shape[0], sr.shape[1]
    out = np.empty((k, S // 2 + 1), dtype=np.float64)
    _load().oracle_trace_spectrum(_p(sr), S, k, _p(out))
    return out


class State:
    """Double-precision simulation state started from the float32 input arrays."""

    def __init__(self, pos_mass, vel, eps2, G):
        pm = np.asarray(pos_mass)
        self.x = np.ascontiguousarray(pm[:, :3].astype(np.float64))
        self.m = np.ascontiguousarray(pm[:, 3].astype(np.float64))
        self.v = np.ascontiguousarray(np.asarray(vel)[:, :3].astype(np.float64))
        self.n = self.x.shape[0]
        self.eps2 = float(eps2)
        self.G = float(G)
        self._work = np.empty_like(self.x)
        self.deformation = None      # (x_psi[3], S) of eq. (10), or None
        self.background = None       # (centre[3], rho_bar), or None

    def step(self, tau, a, H):
        """Eqs. (3)-(5)."""
        if self.deformation is not None or self.background is not None:
            return self.step_coeffs(0.5 * tau, (1.0 - H * tau) / (1.0 + H * tau),
                                    tau / (a ** 3 * (1.0 + H * tau)), 0.5 * tau)
        _load().oracle_step(_p(self.x), _p(self.v), _p(self.m), self.n, self.eps2, self.G,
                            float(tau), float(a), float(H), _p(self._work))

    def step_symplectic(self, cosmo, a0, tau, panels=64, substeps=64):
        """Eq. (9), PAPER.md:64 (reading G11): D(tau/2) K(tau) D(tau/2) in the variable w = a^2 v
        (held in self.v).  Returns a(t + tau)."""
        d1 = int_dt_over_a_pow(cosmo, a0, 0.5 * tau, 2.0, panels)
        a_mid = a_advance(cosmo, a0, 0.5 * tau, substeps)
        d2 = int_dt_over_a_pow(cosmo, a_mid, 0.5 * tau, 2.0, panels)
        ck = int_dt_over_a_pow(cosmo, a0, tau, 1.0, panels)
        self.step_coeffs(d1, 1.0, ck, d2)
        return a_advance(cosmo, a_mid, 0.5 * tau, substeps)

    def step_coeffs(self, d1, cv, ck, d2):
        if self.deformation is not None or self.background is not None:
            xpsi, S = (np.zeros(3), 0.0) if self.deformation is None else \
                (_c64(self.deformation[0]), float(self.deformation[1]))
            cen, rho = (np.zeros(3), 0.0) if self.background is None else \
                (_c64(self.background[0]), float(self.background[1]))
            _load().oracle_step_coeffs_ext(_p(self.x), _p(self.v), _p(self.m), self.n, self.eps2, self.G,
                                           float(d1), float(cv), float(ck), float(d2),
                                           S, _p(xpsi), rho, _p(cen), _p(self._work))
            return
        _load().oracle_step_coeffs(_p(self.x), _p(self.v), _p(self.m), self.n, self.eps2, self.G,
                                   float(d1), float(cv), float(ck), float(d2), _p(self._work))

    def last_force(self):
        """F(x^{n+1/2}) of the most recent step."""
        return self._work.copy()

    def diagnostics(self, a, with_potential=False):
        out = np.zeros(16, dtype=np.float64)
        _load().oracle_diagnostics(_p(self.x), _p(self.v), _p(self.m), self.n, self.eps2, self.G,
                                   float(a), int(bool(with_potential)), _p(out))
        return out


def _cos(c):
    return (float(c.H0), float(c.Om_R), float(c.Om_M), float(c.Om_K), float(c.Om_L))


def hubble(cosmo, a):
    """Eq. (2)."""
    return float(_load().oracle_hubble(*_cos(cosmo), float(a)))


def a_advance(cosmo, a0, dt, substeps=64):
    return float(_load().oracle_a_advance(*_cos(cosmo), float(a0), float(dt), int(substeps)))


def time_of_a(cosmo, a, panels=2_000_000):
    return float(_load().oracle_time_of_a(*_cos(cosmo), float(a), int(panels)))


def int_dt_over_a_pow(cosmo, a0, dt, p, panels=64):
    return float(_load().oracle_int_dt_over_a_pow(*_cos(cosmo), float(a0), float(dt), float(p), int(panels)))


def midstep_schedule(cosmo, a_start, tau, steps, substeps=64):
    """(a, H) at t_n + tau/2 for n = 0..steps-1 (reading G3), plus a at the step ends.

    cosmo None = static background: a = 1, H = 0 (config 3, reading G13)."""
    if cosmo is None:
        return [(1.0, 0.0)] * steps, [1.0] * (steps + 1)
    mids, ends = [], [float(a_start)]
    a = float(a_start)
    for _ in range(steps):
        a_mid = a_advance(cosmo, a, 0.5 * tau, substeps)
        mids.append((a_mid, hubble(cosmo, a_mid)))
        a = a_advance(cosmo, a_mid, 0.5 * tau, substeps)
        ends.append(a)
    return mids, ends
