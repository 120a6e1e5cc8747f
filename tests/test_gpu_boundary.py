"""T1: the C-ABI boundary -- error codes, argument validation, no output on error."""
import numpy as np
import pytest
import ctypes

pytestmark = pytest.mark.gpu

from paper_1208_3444_b200 import binding as B  # noqa: E402


@pytest.fixture()
def session():
    from paper_1208_3444_b200.harness import Session
    s = Session(1.0, 8192)
    yield s
    s.close()


def _code(fn, *args):
    with pytest.raises(B.ColatusError) as e:
        fn(*args)
    return e.value.code


def test_init_twice_and_uninitialised_calls():
    import torch
    assert _code(B.colatus_step, 1e-3, 1.0, 0.0) == B.NOT_INITIALISED
    ws = torch.empty(B.colatus_workspace_bytes(1024), dtype=torch.uint8, device="cuda")
    B.colatus_init(1.0, 0, ws)
    try:
        assert _code(B.colatus_init, 1.0, 0, ws) == B.ALREADY_INITIALISED
        assert _code(B.colatus_step, 1e-3, 1.0, 0.0) == B.NOT_UPLOADED
        assert _code(B.colatus_diagnostics, 1.0) == B.NOT_UPLOADED
        big = torch.zeros((4096, 4), device="cuda")
        assert _code(B.colatus_forces, big, 4096, 1e-4, torch.empty_like(big)) == B.WORKSPACE_TOO_SMALL
    finally:
        B.colatus_shutdown()
    assert _code(B.colatus_forces, ws, 1, 1e-4, ws) == B.NOT_INITIALISED


def test_forces_argument_validation(session):
    import torch
    pm = torch.rand((100, 4), device="cuda")
    out = torch.full((100, 4), 7.0, device="cuda")
    assert _code(B.colatus_forces, None, 100, 1e-4, out) == B.INVALID_ARG
    assert _code(B.colatus_forces, pm, 0, 1e-4, out) == B.INVALID_ARG
    assert _code(B.colatus_forces, pm, 2 ** 31, 1e-4, out) == B.INVALID_ARG
    assert _code(B.colatus_forces, pm, 100, 0.0, out) == B.INVALID_ARG
    assert _code(B.colatus_forces, pm, 100, -1.0, out) == B.INVALID_ARG
    assert _code(B.colatus_forces, pm, 100, float("nan"), out) == B.INVALID_ARG
    assert _code(B.colatus_forces, pm, 100, float("inf"), out) == B.INVALID_ARG
    assert _code(B.colatus_forces, pm, 100, 1e-4, pm) == B.INVALID_ARG                 # aliasing
    assert _code(B.colatus_forces, pm.data_ptr() + 4, 99, 1e-4, out) == B.INVALID_ARG  # misaligned
    assert _code(B.colatus_forces_range, pm, 100, 50, 51, 1e-4, out) == B.INVALID_ARG
    assert _code(B.colatus_forces_range, pm, 100, -1, 10, 1e-4, out) == B.INVALID_ARG
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                                                     # nothing written
    assert "eps2" in B.colatus_last_error() or len(B.colatus_last_error()) > 0


def test_step_argument_validation(session):
    pm = np.random.default_rng(0).random((256, 4)).astype(np.float32)
    vel = np.zeros_like(pm)
    session.upload(pm, vel, 1e-4)
    assert _code(B.colatus_step, float("nan"), 1.0, 0.0) == B.INVALID_ARG
    assert _code(B.colatus_step, 1e-3, 0.0, 0.0) == B.INVALID_ARG
    assert _code(B.colatus_step, 1e-3, -1.0, 0.0) == B.INVALID_ARG
    assert _code(B.colatus_step, 1.0, 1.0, -1.0) == B.INVALID_ARG                      # 1 + H tau = 0
    assert _code(B.colatus_step_coeffs, 1.0, float("inf"), 0.0, 0.0) == B.INVALID_ARG
    assert _code(B.colatus_set_target_range, 200, 100) == B.INVALID_ARG
    assert _code(B.colatus_trace, None, 3, None, 4) == B.INVALID_ARG
    assert _code(B.colatus_trace, None, -1, None, 4) == B.INVALID_ARG
    assert _code(B.colatus_diagnostics, 0.0) == B.INVALID_ARG
    pos, v = session.download()
    assert np.array_equal(pos, pm) and np.array_equal(v, vel)                           # state untouched


def test_nan_inputs_give_nan_outputs_not_errors(session):
    pm = np.random.default_rng(1).random((300, 4)).astype(np.float32)
    pm[7, 0] = np.nan
    out = session.forces(pm, 1e-4).cpu().numpy()
    assert np.isnan(out[:, 0]).all()


def test_launch_count_and_geometry(session):
    pm = np.random.default_rng(2).random((5000, 4)).astype(np.float32)
    c0 = B.colatus_launch_count()
    session.forces(pm, 1e-4)
    geo = B.colatus_force_geometry(5000)
    assert B.colatus_launch_count() - c0 == (2 if geo["source_splits"] == 1 else 3)
    assert geo["sm_count"] == 148 and geo["threads_per_cta"] == 256
    assert geo["target_tiles"] * geo["targets_per_cta"] >= 5000
    assert geo["source_splits"] * geo["sources_per_split"] >= 5000
