"""ctypes binding of libcolatus (include/colatus.h): same names, argument marshalling only.

Device buffers are torch CUDA tensors owned by the caller (PyTorch is used for device memory
and streams only); pointers go through `tensor.data_ptr()` and
`torch.cuda.current_stream().cuda_stream`.  Nothing here computes: no force, no integrator.
If `libcolatus.so` is missing this module raises -- there is no fallback path.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, c_char_p, c_double, c_float, c_int, c_int32, c_int64, c_size_t, c_uint, c_void_p

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcolatus.so")

OK = 0
INVALID_ARG = -1
NOT_INITIALISED = -2
ALREADY_INITIALISED = -3
WORKSPACE_TOO_SMALL = -4
NOT_UPLOADED = -5
UNSUPPORTED_DEVICE = -6
CUDA_ERROR = -7


class ColatusError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"libcolatus error {code}: {text}")
        self.code = code


class colatus_config(Structure):
    _fields_ = [("G", c_double), ("device", c_int), ("workspace_dev", c_void_p),
                ("workspace_bytes", c_size_t), ("flags", c_uint)]


class colatus_cosmo(Structure):
    _fields_ = [("H0", c_double), ("Om_R", c_double), ("Om_M", c_double), ("Om_K", c_double), ("Om_L", c_double)]


# name -> (restype, argtypes): every symbol include/colatus.h declares
SIGNATURES = {
    "colatus_workspace_bytes": (c_size_t, [c_int64]),
    "colatus_init": (c_int, [POINTER(colatus_config)]),
    "colatus_shutdown": (None, []),
    "colatus_forces": (c_int, [c_void_p, c_int64, c_float, c_void_p, c_void_p]),
    "colatus_forces_potential": (c_int, [c_void_p, c_int64, c_float, c_void_p, c_void_p]),
    "colatus_forces_range": (c_int, [c_void_p, c_int64, c_int64, c_int64, c_float, c_void_p, c_void_p]),
    "colatus_forces_host": (c_int, [c_void_p, c_int64, c_float, c_void_p, c_void_p]),
    "colatus_forces_static": (c_int, [c_void_p, c_int64, c_float, c_double, c_void_p, c_void_p]),
    "colatus_upload": (c_int, [c_void_p, c_void_p, c_void_p, c_int64, c_float, c_void_p]),
    "colatus_step": (c_int, [c_double, c_double, c_double]),
    "colatus_step_coefficients": (c_int, [c_double, c_double, c_double, POINTER(c_double)]),
    "colatus_step_coeffs": (c_int, [c_double, c_double, c_double, c_double]),
    "colatus_run": (c_int, [POINTER(colatus_cosmo), c_double, c_double, c_int64, c_int, POINTER(c_double)]),
    "colatus_run_symplectic": (c_int, [POINTER(colatus_cosmo), c_double, c_double, c_int64, c_int, POINTER(c_double)]),
    "colatus_symplectic_coefficients": (c_int, [POINTER(colatus_cosmo), c_double, c_double, POINTER(c_double)]),
    "colatus_step_symplectic": (c_int, [POINTER(colatus_cosmo), c_double, c_double, POINTER(c_double)]),
    "colatus_set_deformation": (c_int, [POINTER(c_double), c_double]),
    "colatus_set_background": (c_int, [POINTER(c_double), c_double]),
    "colatus_set_target_range": (c_int, [c_int64, c_int64]),
    "colatus_drift": (c_int, [c_double]),
    "colatus_force_kick_drift": (c_int, [c_double, c_double, c_double]),
    "colatus_kick_drift": (c_int, [c_void_p, c_double, c_double, c_double]),
    "colatus_add_external": (c_int, [c_void_p]),
    "colatus_forces_symmetric_part": (c_int, [c_void_p, c_int64, c_float, c_int, c_int, c_void_p, c_void_p]),
    "colatus_trace": (c_int, [c_void_p, c_int, c_void_p, c_int]),
    "colatus_trace_read": (c_int, [c_void_p, c_int64, c_int]),
    "colatus_splat": (c_int, [c_void_p, c_int64, c_int, POINTER(c_float), c_int, c_int, c_void_p, c_void_p]),
    "colatus_trace_spectrum": (c_int, [c_int64, c_int, c_void_p]),
    "colatus_diagnostics": (c_int, [c_double, c_int, POINTER(c_double)]),
    "colatus_download": (c_int, [c_void_p, c_void_p]),
    "colatus_profile": (c_int, [c_int]),
    "colatus_profile_read": (c_int, [POINTER(c_double), POINTER(c_int64)]),
    "colatus_launch_count": (c_int64, []),
    "colatus_force_geometry": (c_int, [c_int64, c_int64, POINTER(c_int64)]),
    "colatus_force_plan": (c_int, [c_int64, c_int64, c_int, POINTER(c_int64)]),
    "colatus_set_option": (c_int, [c_char_p, c_int64]),
    "colatus_last_error": (c_char_p, []),
    "colatus_hubble": (c_double, [POINTER(colatus_cosmo), c_double]),
    "colatus_a_advance": (c_double, [POINTER(colatus_cosmo), c_double, c_double]),
    "colatus_time_of_a": (c_double, [POINTER(colatus_cosmo), c_double]),
    "colatus_int_dt_over_a_pow": (c_double, [POINTER(colatus_cosmo), c_double, c_double, c_double]),
}

_lib = None


def lib():
    """Load libcolatus.so (built in-tree by `paper_1208_3444_b200.build`); raise if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ColatusError(CUDA_ERROR, f"{LIB_PATH} is missing: run `python -m paper_1208_3444_b200.build` "
                                           "(there is no CPU fallback)")
        handle = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(handle, name)
            fn.restype = res
            fn.argtypes = args
        _lib = handle
    return _lib


def _check(rc):
    if rc != OK:
        raise ColatusError(rc, lib().colatus_last_error().decode())


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream


def _ptr(t):
    return None if t is None else (t if isinstance(t, int) else t.data_ptr())


# ---- host-only cosmology (eq. 2) -------------------------------------------------------------
def _cosmo(c):
    return colatus_cosmo(float(c.H0), float(c.Om_R), float(c.Om_M), float(c.Om_K), float(c.Om_L))


def colatus_hubble(cosmo, a):
    return lib().colatus_hubble(ctypes.byref(_cosmo(cosmo)), float(a))


def colatus_a_advance(cosmo, a0, dt):
    return lib().colatus_a_advance(ctypes.byref(_cosmo(cosmo)), float(a0), float(dt))


def colatus_time_of_a(cosmo, a):
    return lib().colatus_time_of_a(ctypes.byref(_cosmo(cosmo)), float(a))


def colatus_int_dt_over_a_pow(cosmo, a0, dt, p):
    return lib().colatus_int_dt_over_a_pow(ctypes.byref(_cosmo(cosmo)), float(a0), float(dt), float(p))


# ---- device entry points ---------------------------------------------------------------------
def colatus_workspace_bytes(n_max):
    return int(lib().colatus_workspace_bytes(int(n_max)))


def colatus_init(G, device, workspace, flags=0):
    """`workspace`: a torch.uint8 CUDA tensor of >= colatus_workspace_bytes(n_max) bytes."""
    cfg = colatus_config(float(G), int(device), workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                         int(flags))
    _check(lib().colatus_init(ctypes.byref(cfg)))


def colatus_shutdown():
    lib().colatus_shutdown()


def colatus_forces(pos_mass, n, eps2, acc_out, stream=None):
    _check(lib().colatus_forces(_ptr(pos_mass), int(n), float(eps2), _ptr(acc_out), _stream(stream)))


def colatus_forces_potential(pos_mass, n, eps2, acc_out, stream=None):
    _check(lib().colatus_forces_potential(_ptr(pos_mass), int(n), float(eps2), _ptr(acc_out), _stream(stream)))


def colatus_forces_range(pos_mass, n, target_begin, target_count, eps2, acc_out, stream=None):
    _check(lib().colatus_forces_range(_ptr(pos_mass), int(n), int(target_begin), int(target_count), float(eps2),
                                      _ptr(acc_out), _stream(stream)))


def colatus_forces_symmetric_part(pos_mass, n, eps2, part, parts, acc_out, stream=None):
    _check(lib().colatus_forces_symmetric_part(_ptr(pos_mass), int(n), float(eps2), int(part), int(parts),
                                               _ptr(acc_out), _stream(stream)))


def colatus_forces_host(pos_mass_host, n, eps2, acc_out_host, stream=None):
    """Host buffers: numpy float32 arrays or pinned torch CPU tensors of shape [n,4]."""
    _check(lib().colatus_forces_host(_host_ptr(pos_mass_host), int(n), float(eps2), _host_ptr(acc_out_host),
                                     _stream(stream)))


STATIC_MAX_N = 32768          # COLATUS_STATIC_MAX_N of include/colatus.h


def colatus_forces_static(pos_mass, n, eps2, G, acc_out, stream=None):
    """Eq. (1) for callers who cannot cudaMalloc a workspace (a plug-in under another allocator, a loop that must
    not synchronise the device): scratch lives in an array inside libcolatus, so n <= STATIC_MAX_N.  Needs no
    colatus_init; runs on the current device.  Calls share that array: keep them ordered on the GPU."""
    _check(lib().colatus_forces_static(_ptr(pos_mass), int(n), float(eps2), float(G), _ptr(acc_out), _stream(stream)))


def _host_ptr(a):
    if a is None:
        return None
    if hasattr(a, "ctypes"):
        return a.ctypes.data
    return a.data_ptr()


def colatus_upload(pos_mass, vel, acc, n, eps2, stream=None):
    _check(lib().colatus_upload(_ptr(pos_mass), _ptr(vel), _ptr(acc), int(n), float(eps2), _stream(stream)))


def colatus_step(tau, a, H):
    _check(lib().colatus_step(float(tau), float(a), float(H)))


def colatus_step_coefficients(tau, a, H):
    out = (c_double * 4)()
    _check(lib().colatus_step_coefficients(float(tau), float(a), float(H), out))
    return tuple(out)


def colatus_step_coeffs(d1, cv, ck, d2):
    _check(lib().colatus_step_coeffs(float(d1), float(cv), float(ck), float(d2)))


def colatus_run(cosmo, a_start, tau, n_steps, use_graph=True):
    """n_steps steps of eqs. (3)-(5) in one native call (CUDA-graph replay); cosmo None = static.  Returns a_end."""
    a_end = c_double(0.0)
    cp = None if cosmo is None else ctypes.byref(_cosmo(cosmo))
    _check(lib().colatus_run(cp, float(a_start), float(tau), int(n_steps), int(bool(use_graph)), ctypes.byref(a_end)))
    return a_end.value


def colatus_run_symplectic(cosmo, a_start, tau, n_steps, use_graph=True):
    """n_steps symplectic steps of eq. (9) in one native call (CUDA-graph replay).  Returns a_end."""
    a_end = c_double(0.0)
    cp = None if cosmo is None else ctypes.byref(_cosmo(cosmo))
    _check(lib().colatus_run_symplectic(cp, float(a_start), float(tau), int(n_steps), int(bool(use_graph)),
                                        ctypes.byref(a_end)))
    return a_end.value


def colatus_symplectic_coefficients(cosmo, a0, tau):
    """Eq. (9): (d1, cv = 1, ck, d2, a_end), host only."""
    out = (c_double * 5)()
    _check(lib().colatus_symplectic_coefficients(ctypes.byref(_cosmo(cosmo)), float(a0), float(tau), out))
    return tuple(out)


def colatus_step_symplectic(cosmo, a0, tau):
    """One symplectic drift-kick-drift step of eq. (9); returns a(t + tau)."""
    a_end = c_double(0.0)
    _check(lib().colatus_step_symplectic(ctypes.byref(_cosmo(cosmo)), float(a0), float(tau), ctypes.byref(a_end)))
    return a_end.value


def colatus_set_deformation(x_psi, strength):
    """Eq. (10): fixed source of strength S = C*psi at x_psi; strength 0 disables."""
    v = (c_double * 3)(*[float(c) for c in (x_psi if x_psi is not None else (0, 0, 0))])
    _check(lib().colatus_set_deformation(v, float(strength)))


def colatus_set_background(centre, rho_bar):
    """Mean-density background term (reading G22); rho_bar 0 disables."""
    v = (c_double * 3)(*[float(c) for c in (centre if centre is not None else (0, 0, 0))])
    _check(lib().colatus_set_background(v, float(rho_bar)))


def colatus_set_target_range(begin, count):
    _check(lib().colatus_set_target_range(int(begin), int(count)))


def colatus_drift(d):
    _check(lib().colatus_drift(float(d)))


def colatus_force_kick_drift(cv, ck, d2):
    _check(lib().colatus_force_kick_drift(float(cv), float(ck), float(d2)))


def colatus_kick_drift(acc, cv, ck, d2):
    _check(lib().colatus_kick_drift(_ptr(acc), float(cv), float(ck), float(d2)))


def colatus_add_external(acc):
    """Adds the eq. (10) source / background term once to caller-assembled forces of the resident target range."""
    _check(lib().colatus_add_external(_ptr(acc)))


def colatus_trace(idx, k, ring, capacity_steps):
    _check(lib().colatus_trace(_ptr(idx), int(k), _ptr(ring), int(capacity_steps)))


def colatus_trace_read(host_out, first_step, n_steps):
    _check(lib().colatus_trace_read(_host_ptr(host_out), int(first_step), int(n_steps)))


def colatus_splat(pos_mass, n, axis, window, width, height, image, stream=None):
    """Particle-count image (Fig. 1); pos_mass None = resident state."""
    win = (c_float * 6)(*[float(c) for c in window])
    _check(lib().colatus_splat(None if pos_mass is None else _ptr(pos_mass), int(n), int(axis), win,
                               int(width), int(height), _ptr(image), _stream(stream)))


def colatus_trace_spectrum(first_step, n_steps, spectrum):
    """Periodogram of the tracer velocity series into a device double [k, n_steps//2+1]."""
    _check(lib().colatus_trace_spectrum(int(first_step), int(n_steps), _ptr(spectrum)))


def colatus_diagnostics(a, with_potential=False):
    out = (c_double * 16)()
    _check(lib().colatus_diagnostics(float(a), int(bool(with_potential)), out))
    return list(out)


def colatus_download(pos_mass_host=None, vel_host=None):
    _check(lib().colatus_download(_host_ptr(pos_mass_host), _host_ptr(vel_host)))


def colatus_profile(enable):
    _check(lib().colatus_profile(int(bool(enable))))


def colatus_profile_read():
    ms, k = c_double(0.0), c_int64(0)
    _check(lib().colatus_profile_read(ctypes.byref(ms), ctypes.byref(k)))
    return ms.value, k.value


def colatus_launch_count():
    return int(lib().colatus_launch_count())


def colatus_force_geometry(n, target_count=None):
    out = (c_int64 * 8)()
    _check(lib().colatus_force_geometry(int(n), int(n if target_count is None else target_count), out))
    keys = ("targets_per_cta", "target_tiles", "source_splits", "sources_per_split", "ctas_per_sm", "sm_count",
            "targets_per_thread", "threads_per_cta")
    return dict(zip(keys, [int(v) for v in out]))


def colatus_force_plan(n, target_count=None, with_potential=False):
    out = (c_int64 * 8)()
    _check(lib().colatus_force_plan(int(n), int(n if target_count is None else target_count),
                                    1 if with_potential else 0, out))
    keys = ("symmetric", "blocks", "splits", "distances", "distances_per_launch", "launches", "padded_bodies",
            "partial_rows")
    return dict(zip(keys, [int(v) for v in out]))


def colatus_set_option(name, value):
    _check(lib().colatus_set_option(name.encode(), int(value)))


def colatus_last_error():
    return lib().colatus_last_error().decode()
