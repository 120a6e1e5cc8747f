"""colatus_run: the native step loop with a device coefficient table and CUDA-graph replay must be bitwise
identical to calling colatus_step once per step from the host (same kernels' arithmetic, same FP64 schedule
of eq. (2)), and hence inherits the oracle parity of tests/test_gpu_steps.py; it is also checked against the
oracle directly."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_1208_3444_b200 import binding as B  # noqa: E402
from paper_1208_3444_b200 import inputs  # noqa: E402

POS_TOL = 1e-5


def _session(G, n):
    from paper_1208_3444_b200.harness import Session
    return Session(G, n)


def _run(cfg, pm, vel, steps, mode, tracers=None, capacity=None):
    with _session(cfg.G, cfg.n) as s:
        s.upload(pm, vel, cfg.eps2)
        if tracers is not None:
            s.trace(tracers, capacity)
        if mode == "host":
            a_end = s.run(cfg.cosmo, cfg.a_start, cfg.tau, steps)
        else:
            a_end = s.run_native(cfg.cosmo, cfg.a_start, cfg.tau, steps, use_graph=(mode == "graph"))
        pos, v = s.download()
        diag = s.diagnostics(1.0)
        ring = s.ring.cpu().numpy() if tracers is not None else None
    return a_end, pos, v, diag, ring


@pytest.mark.parametrize("index,n_override,steps", [(1, None, 12), (2, 4913, 7), (3, 9001, 6), (3, 100, 9), (1, 2, 5)])
def test_run_equals_step_loop_bitwise(index, n_override, steps):
    cfg, pm, vel = inputs.make_config(index, n_override)
    rng = np.random.Generator(np.random.PCG64(9))
    vel = vel.copy()
    vel[:, :3] = 0.01 * rng.standard_normal((cfg.n, 3)).astype(np.float32)
    tracers = np.arange(0, cfg.n, max(cfg.n // 16, 1), dtype=np.int32)[:16]
    ref = _run(cfg, pm, vel, steps, "host", tracers, 5)               # ring of 5 rows wraps
    for mode in ("graph", "launch"):
        got = _run(cfg, pm, vel, steps, mode, tracers, 5)
        assert got[0] == ref[0]
        assert np.array_equal(got[1], ref[1]) and np.array_equal(got[2], ref[2])
        assert got[3][12] == steps
        assert np.array_equal(got[4], ref[4])


def test_run_against_oracle_config1():
    cfg, pm, vel = inputs.make_config(1)
    steps = cfg.parity_steps
    a_end, pos, _, _, _ = _run(cfg, pm, vel, steps, "graph")
    st = oracle.State(pm, vel, cfg.eps2, cfg.G)
    mids, ends = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, steps)
    for a, H in mids:
        st.step(cfg.tau, a, H)
    assert a_end == pytest.approx(ends[-1], rel=1e-9)
    assert np.linalg.norm(pos[:, :3].astype(np.float64) - st.x, axis=1).max() <= POS_TOL


def test_run_many_steps_table_chunks_and_split_calls():
    """2500 static steps of a small system cross two table uploads (1024 steps each); splitting the run into
    several calls, with graph and without, changes nothing."""
    cfg, pm, vel = inputs.make_config(3, n_override=300)
    tr = np.array([0, 150, 299], dtype=np.int32)
    outs = []
    for plan in ([(2500, True)], [(1000, False), (24, True), (1476, True)], [(2500, False)]):
        with _session(cfg.G, cfg.n) as s:
            s.upload(pm, vel, cfg.eps2)
            s.trace(tr, 4096)
            for n_steps, graph in plan:
                s.run_native(None, 1.0, 2e-4, n_steps, use_graph=graph)
            pos, v = s.download()
            rows = s.trace_read(0, 2500)
            outs.append((pos, v, rows, s.diagnostics(1.0)[12]))
    for o in outs[1:]:
        assert np.array_equal(o[0], outs[0][0]) and np.array_equal(o[1], outs[0][1]) and np.array_equal(o[2], outs[0][2])
        assert o[3] == 2500
    assert np.abs(outs[0][0][:, :3] - pm[:, :3]).max() > 1e-3        # it did move


def test_run_graph_recaptured_after_state_changes():
    """The cached graph bakes in the target range, tracer set and external terms: each change re-captures."""
    cfg, pm, vel = inputs.make_config(1)

    def sequence(native):
        with _session(cfg.G, cfg.n) as s:
            s.upload(pm, vel, cfg.eps2)
            step = (lambda k: s.run_native(None, 1.0, 1e-3, k)) if native else (lambda k: s.run(None, 1.0, 1e-3, k))
            step(2)
            B.colatus_set_target_range(1000, 2000)
            step(2)
            B.colatus_set_target_range(0, cfg.n)
            s.trace(np.array([5, 7], dtype=np.int32), 8)
            step(2)
            B.colatus_set_deformation((0.5, 0.5, 1.5), 0.2)
            step(2)
            B.colatus_set_deformation(None, 0.0)
            B.colatus_set_option("source_splits", 3)
            step(1)
            B.colatus_set_option("source_splits", 0)
            pos, v = s.download()
            return pos, v, s.ring.cpu().numpy()

    a, b = sequence(False), sequence(True)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


def test_run_argument_validation_enqueues_nothing():
    cfg, pm, vel = inputs.make_config(1)
    with _session(cfg.G, cfg.n) as s:
        with pytest.raises(B.ColatusError):
            B.colatus_run(cfg.cosmo, cfg.a_start, cfg.tau, 3)          # not uploaded
        s.upload(pm, vel, cfg.eps2)
        for args in ((cfg.cosmo, cfg.a_start, cfg.tau, 0), (cfg.cosmo, -1.0, cfg.tau, 3),
                     (cfg.cosmo, cfg.a_start, float("nan"), 3), (cfg.cosmo, cfg.a_start, -1.0, 3)):   # 1 + H tau <= 0
            with pytest.raises(B.ColatusError):
                B.colatus_run(*args)
        pos, v = s.download()
        assert np.array_equal(pos, pm) and np.array_equal(v, vel) and s.diagnostics(1.0)[12] == 0


def test_cached_graph_honours_a_mass_change_between_runs():
    """The equal-mass decision is taken on the device at every force evaluation (stage kernel stamps a flag),
    so a graph captured while all masses were equal stays correct after the caller edits a mass in its
    resident buffer -- bitwise the same as per-step colatus_step calls on the same sequence."""
    import torch
    cfg, pm, vel = inputs.make_config(1)
    outs = []
    for native in (True, False):
        from paper_1208_3444_b200.harness import Session
        with Session(cfg.G, cfg.n) as s:
            s.upload(pm, vel, cfg.eps2)
            step = (lambda k: s.run_native(None, 1.0, 1e-3, k)) if native else (lambda k: s.run(None, 1.0, 1e-3, k))
            step(3)
            torch.cuda.synchronize()
            s.pos[100, 3] *= 40.0                      # the caller owns the buffer
            step(3)
            s.pos[100, 3] /= 40.0
            step(2)
            outs.append(s.download())
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    st = oracle.State(pm, vel, cfg.eps2, cfg.G)
    for k in range(8):
        st.m[100] = pm[100, 3] * (40.0 if 3 <= k < 6 else 1.0)
        st.step(1e-3, 1.0, 0.0)
    assert np.linalg.norm(outs[0][0][:, :3].astype(np.float64) - st.x, axis=1).max() <= POS_TOL


@pytest.mark.parametrize("use_graph", [True, False])
def test_run_symplectic_equals_step_symplectic_loop_bitwise(use_graph):
    """Eq. (9) in the native loop: same coefficients, same kernels as colatus_step_symplectic per step."""
    cfg, pm, vel = inputs.make_config(1)
    rng = np.random.Generator(np.random.PCG64(21))
    w0 = vel.copy()
    w0[:, :3] = (cfg.a_start ** 2) * 0.05 * rng.standard_normal((cfg.n, 3)).astype(np.float32)
    tr = np.arange(0, cfg.n, 256, dtype=np.int32)
    outs = []
    from paper_1208_3444_b200.harness import Session
    for native in (False, True):
        with Session(cfg.G, cfg.n) as s:
            s.upload(pm, w0, cfg.eps2)
            s.trace(tr, 4)
            a = cfg.a_start
            if native:
                a = B.colatus_run_symplectic(cfg.cosmo, a, cfg.tau, 6, use_graph)
            else:
                for _ in range(6):
                    a = B.colatus_step_symplectic(cfg.cosmo, a, cfg.tau)
            pos, w = s.download()
            outs.append((a, pos, w, s.ring.cpu().numpy()))
    assert outs[0][0] == outs[1][0]
    for x, y in zip(outs[0][1:], outs[1][1:]):
        assert np.array_equal(x, y)
    st = oracle.State(pm, w0, cfg.eps2, cfg.G)
    a_ref = cfg.a_start
    for _ in range(6):
        a_ref = st.step_symplectic(cfg.cosmo, a_ref, cfg.tau)
    assert outs[1][0] == pytest.approx(a_ref, rel=1e-9)
    assert np.linalg.norm(outs[1][1][:, :3].astype(np.float64) - st.x, axis=1).max() <= POS_TOL
