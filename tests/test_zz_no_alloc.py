"""colatus_forces_static (include/colatus.h): eq. (1), for callers who cannot allocate device memory.

Who that is: code that runs inside somebody else's application and must live with the device memory it is handed
(the host's own pool has taken the rest), a control loop or callback that cannot afford cudaMalloc's device-wide
synchronisation or a late out-of-memory error, a job with a fixed device-memory budget.  Such a caller cannot
provide the workspace every other entry point needs, so this one keeps its scratch in an array that is part of
libcolatus' device image (4.5 MiB, good for n <= COLATUS_STATIC_MAX_N = 32768) and needs no colatus_init.

What is checked here, on a GPU:
  * its forces against those of the existing workspace path (colatus_forces) on the same inputs, within the
    tolerances the force tests use (test_gpu_forces.py: median relative error 1e-5, max over rms 1e-4) -- on
    calls made back to back WITHOUT synchronising in between, of different sizes and mass kinds, because every
    call reuses the one array and finds in it whatever the call before left (a stale equal-mass flag or stale
    partial sums would show up in exactly this sequence);
  * that a repeated call returns the same bits, that sizes beyond the limit are refused with a message naming
    the limit and leave the output alone, and that the calls leave the device's free memory where it was.

The file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here
must not hide the rest of the suite.  It passes alone in a fresh process (the first static call then precedes
any colatus_init) and after the other GPU tests (the library context is then already shut down again).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1208_3444_b200 import binding as B  # noqa: E402

MEDIAN_TOL = 1e-5      # as tests/test_gpu_forces.py (north_star, reading G17)
MAX_TOL = 1e-4
G = 0.75               # not 1: the static entry point takes G as an argument and has to apply it


def _force_errors(got, ref):
    d = np.linalg.norm(got.astype(np.float64) - ref.astype(np.float64), axis=1)
    nr = np.linalg.norm(ref.astype(np.float64), axis=1)
    return float(np.median(d / nr)), float(d.max() / np.sqrt((nr ** 2).mean()))


def _problem(n, equal_mass, seed):
    """Half uniform in the unit box, half in a tight clump (close pairs), shuffled; equal or log-normal masses."""
    rng = np.random.Generator(np.random.PCG64(77100 + seed))
    pm = np.empty((n, 4), dtype=np.float32)
    half = n // 2
    pm[:half, :3] = rng.random((half, 3))
    pm[half:, :3] = 0.5 + 0.03 * rng.standard_normal((n - half, 3))
    pm[:, 3] = 1.0 / n if equal_mass else np.exp(0.5 * rng.standard_normal(n)) / n
    return pm[rng.permutation(n)]


# (n, equal masses): the paper's 32^3 with equal masses first, then a smaller ragged problem with unequal masses
# (it must not see the flag or the partial sums of the first), then equal masses again (the flag must be cleared)
CALLS = [(B.STATIC_MAX_N, True), (5003, False), (20000, True), (1, True), (777, False)]


def test_static_forces_match_the_workspace_path_on_consecutive_calls():
    import torch
    from paper_1208_3444_b200.harness import Session

    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    eps2 = np.float32(1e-4)
    problems = [_problem(n, eq, seed=i) for i, (n, eq) in enumerate(CALLS)]
    pms = [torch.from_numpy(p).to(dev) for p in problems]
    outs = [torch.full((p.shape[0], 4), float("nan"), dtype=torch.float32, device=dev) for p in problems]
    again = torch.full((problems[0].shape[0], 4), float("nan"), dtype=torch.float32, device=dev)

    # first call on this device: does the one-time set-up (and, in a fresh process, comes before any colatus_init)
    B.colatus_forces_static(pms[0], problems[0].shape[0], eps2, G, outs[0])
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]

    # the calls in a row, one stream, no synchronisation between them
    for pm, p, out in zip(pms, problems, outs):
        B.colatus_forces_static(pm, p.shape[0], eps2, G, out)
    B.colatus_forces_static(pms[0], problems[0].shape[0], eps2, G, again)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "colatus_forces_static must not take device memory"
    static = [o.cpu().numpy() for o in outs]
    assert np.array_equal(static[0], again.cpu().numpy()), "same input after other calls: same bits"

    # the existing path: a workspace somebody allocated, colatus_init, colatus_forces
    with Session(G, B.STATIC_MAX_N) as s:
        for (n, eq), pm, got in zip(CALLS, pms, static):
            ref = s.forces(pm, eps2).cpu().numpy()
            assert np.all(got[:, 3] == 0.0)
            if n == 1:
                assert np.all(got == 0.0) and np.all(ref == 0.0)
                continue
            assert np.isfinite(got).all()
            med, mx = _force_errors(got[:, :3], ref[:, :3])
            assert med <= MEDIAN_TOL and mx <= MAX_TOL, (n, eq, med, mx)
        # mixing is allowed: a static call while the workspace path is initialised changes neither
        B.colatus_forces_static(pms[1], problems[1].shape[0], eps2, G, again[:problems[1].shape[0]])
        torch.cuda.synchronize()
        assert np.array_equal(again[:problems[1].shape[0]].cpu().numpy(), static[1])


def test_static_forces_refuse_what_the_array_cannot_hold():
    import torch

    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    n = B.STATIC_MAX_N + 1
    pm = torch.from_numpy(_problem(n, True, seed=99)).to(dev)
    out = torch.full((n, 4), 7.0, dtype=torch.float32, device=dev)
    with pytest.raises(B.ColatusError) as e:
        B.colatus_forces_static(pm, n, 1e-4, G, out)
    assert e.value.code == B.INVALID_ARG
    assert "COLATUS_STATIC_MAX_N" in str(e.value) and str(B.STATIC_MAX_N) in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all()), "a refused call writes nothing"
    for bad_n in (0, -3):
        with pytest.raises(B.ColatusError):
            B.colatus_forces_static(pm, bad_n, 1e-4, G, out)
    with pytest.raises(B.ColatusError):
        B.colatus_forces_static(pm, 100, 0.0, G, out)              # eps2 below the floor
    with pytest.raises(B.ColatusError):
        B.colatus_forces_static(pm, 100, 1e-4, float("inf"), out)  # G not finite
    with pytest.raises(B.ColatusError):
        B.colatus_forces_static(pm, 100, 1e-4, G, pm)              # aliasing
