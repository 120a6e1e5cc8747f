"""The target-sharded driver (paper_1208_3444_b200/sharded.py) on the GPU through the C ABI:
ShardedStepper + LibcolatusOps at world size 1 (no process group -- one GPU is all this box has) must reproduce
the oracle's trajectory, diagnostics and tracer record like the single-GPU path does.  The exchange step itself
(all-gather / all-reduce sequencing at world size 2) is covered on CPU by tests/test_sharded_gloo.py."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_1208_3444_b200 import binding as B  # noqa: E402
from paper_1208_3444_b200 import inputs  # noqa: E402


def test_sharded_stepper_world1_matches_oracle():
    import torch
    from paper_1208_3444_b200.harness import Session
    from paper_1208_3444_b200.sharded import LibcolatusOps, ShardedStepper
    cfg, pm, vel = inputs.make_config(1)
    steps = 10
    tr = np.arange(0, cfg.n, cfg.n // 16, dtype=np.int32)
    with Session(cfg.G, cfg.n) as s:
        pos, v = s.to_device(pm), s.to_device(vel)
        acc = torch.zeros_like(pos)
        ops = LibcolatusOps(pos, v, acc, cfg.n, cfg.eps2, 0, cfg.n)
        stepper = ShardedStepper(pos, cfg.n, ops)
        assert (stepper.world, stepper.begin, stepper.count) == (1, 0, cfg.n)
        idx = torch.from_numpy(tr).to(pos.device)
        ring = torch.zeros((steps, tr.size, 4), dtype=torch.float32, device=pos.device)
        ops.trace(idx, ring, steps)
        mids, ends = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, steps)
        for a, H in mids:
            stepper.step(cfg.tau, a, H)
        assert stepper.gathers == 0 and not stepper.dirty
        d = stepper.diagnostics(ends[-1], with_potential=True)
        rows = stepper.trace_read(tr, 0, steps)
        torch.cuda.synchronize()
        x_gpu, v_gpu = pos.cpu().numpy(), v.cpu().numpy()
    st = oracle.State(pm, vel, cfg.eps2, cfg.G)
    rows_ref = np.zeros((steps, tr.size, 3))
    for n, (a, H) in enumerate(mids):
        st.step(cfg.tau, a, H)
        rows_ref[n] = st.v[tr]
    assert np.linalg.norm(x_gpu[:, :3].astype(np.float64) - st.x, axis=1).max() <= 1e-5          # G16
    dref = st.diagnostics(ends[-1], with_potential=True)
    assert d[0] == pytest.approx(dref[0], rel=1e-6) and d[7] == pytest.approx(dref[7], rel=1e-4)
    assert d[8] == pytest.approx(dref[8], rel=1e-5) and d[12] == steps
    assert np.allclose(d[9:12], dref[9:12], atol=2e-6) and np.allclose(d[13:16], d[9:12] * d[0], rtol=1e-12)
    assert np.array_equal(rows[-1, :, :3], v_gpu[tr, :3])                                        # bit-exact record
    vr = np.sqrt((rows_ref ** 2).sum(2).mean())
    assert np.abs(rows[:, :, :3] - rows_ref).max() <= 2e-4 * vr


def test_sharded_two_slices_evaluated_one_after_the_other_equal_the_full_step():
    """What rank 0 and rank 1 of a 2-GPU run would each compute, done one after the other on this GPU (no
    kernel waits on another): drift / force-kick-drift restricted to a slice touch that slice only, and the two
    slices together equal the unsharded step up to the summation order (the source split is chosen per target
    count, reading G14)."""
    import torch
    from paper_1208_3444_b200.harness import Session
    cfg, pm, vel = inputs.make_config(1)
    rng = np.random.Generator(np.random.PCG64(5))
    vel = vel.copy()
    vel[:, :3] = 0.05 * rng.standard_normal((cfg.n, 3)).astype(np.float32)
    c = B.colatus_step_coefficients(cfg.tau, 0.05, 3.0)
    half = cfg.n // 2
    with Session(cfg.G, cfg.n) as s:
        # reference: whole range through the same separate kernels (drift, force, kick-drift)
        s.upload(pm, vel, cfg.eps2)
        B.colatus_set_target_range(0, cfg.n)
        B.colatus_drift(c[0])
        B.colatus_force_kick_drift(c[1], c[2], c[3])
        x_ref, v_ref = s.download()
        # "two ranks": both drift their slice of the same start state, the drifted slices are exchanged
        # (here: they already sit in the one array), then each force-kick-drifts its slice from a copy of the
        # gathered positions
        s.upload(pm, vel, cfg.eps2)
        for b in (0, half):
            B.colatus_set_target_range(b, half)
            B.colatus_drift(c[0])
        torch.cuda.synchronize()
        gathered = s.pos.clone()
        out_x, out_v = np.empty_like(pm), np.empty_like(vel)
        for b in (0, half):
            s.pos.copy_(gathered)
            acc = torch.zeros((half, 4), dtype=torch.float32, device=s.pos.device)
            B.colatus_upload(s.pos, s.vel, acc, cfg.n, cfg.eps2)
            B.colatus_set_target_range(b, half)
            B.colatus_force_kick_drift(c[1], c[2], c[3])
            x, v = s.download()
            other = slice(half, cfg.n) if b == 0 else slice(0, half)
            assert np.array_equal(x[other], gathered.cpu().numpy()[other])          # other slice untouched
            out_x[b:b + half], out_v[b:b + half] = x[b:b + half], v[b:b + half]
            s.vel.copy_(s.to_device(vel))                                            # rank-local velocities
    assert np.array_equal(out_x[:, 3], x_ref[:, 3])
    vr = float(np.sqrt((v_ref[:, :3].astype(np.float64) ** 2).sum(1).mean()))
    assert np.abs(out_v[:, :3] - v_ref[:, :3]).max() <= 2e-5 * vr
    assert np.abs(out_x[:, :3] - x_ref[:, :3]).max() <= 1e-6
    assert not np.array_equal(out_x[:, :3], pm[:, :3])


# ---- the symmetric evaluation divided over GPUs (colatus_forces_symmetric_part; sharded.py symmetric mode) ---------
@pytest.mark.parametrize("block", [1024, 1536, 4096])
@pytest.mark.parametrize("parts", [1, 2, 3, 5, 8])
def test_symmetric_parts_add_up_to_the_whole_force(parts, block):
    """Each share of the block pairs, evaluated on this GPU one after the other (what the ranks of a `parts`-GPU run
    compute at the same time): the partial forces on ALL bodies add up to the oracle's forces; shares of different
    sizes (blocks not divisible by parts), even and odd block counts, chunked block distances."""
    import torch
    from paper_1208_3444_b200.harness import Session
    cfg, pm, _ = inputs.make_config(4, n_override=21000)            # log-normal masses, clusters
    ref = oracle.forces(pm, cfg.eps2, 1.0)
    rms = np.sqrt((ref ** 2).sum(1).mean())
    with Session(1.0, cfg.n) as s:
        B.colatus_set_option("symmetric_block", block)
        pm_d = s.to_device(pm)
        for rows in (0, 7):
            B.colatus_set_option("symmetric_rows", rows)
            total = np.zeros((cfg.n, 3))
            reached = np.zeros(cfg.n, dtype=bool)
            for part in range(parts):
                out = torch.full((cfg.n, 4), np.nan, dtype=torch.float32, device=pm_d.device)
                B.colatus_forces_symmetric_part(pm_d, cfg.n, cfg.eps2, part, parts, out)
                o = out.cpu().numpy()
                assert np.isfinite(o).all() and np.all(o[:, 3] == 0.0)
                total += o[:, :3].astype(np.float64)
                reached |= np.any(o[:, :3] != 0.0, axis=1)
            assert reached.all()
            d = np.linalg.norm(total - ref, axis=1)
            assert np.median(d / np.linalg.norm(ref, axis=1)) <= 1e-5 and d.max() / rms <= 1e-4, (parts, block, rows)
        with pytest.raises(B.ColatusError):
            B.colatus_forces_symmetric_part(pm_d, cfg.n, cfg.eps2, parts, parts, out)


def test_symmetric_shares_are_disjoint_in_what_they_own():
    """With 14 shares of 14 blocks (H = 6) share 0 is block 0: it delivers to itself (its own sums, incl. the
    one-directional term of the antipodal block 7 acting on IT) and reactions to the 6 blocks after it; every other
    body gets exactly 0 from it (the all-reduce adds exact zeros there)."""
    import torch
    from paper_1208_3444_b200.harness import Session
    cfg, pm, _ = inputs.make_config(3, n_override=14 * 1536)
    with Session(1.0, cfg.n) as s:
        B.colatus_set_option("symmetric_block", 1536)
        pm_d = s.to_device(pm)
        out = torch.empty((cfg.n, 4), dtype=torch.float32, device=pm_d.device)
        B.colatus_forces_symmetric_part(pm_d, cfg.n, cfg.eps2, 0, 14, out)       # share 0 = block 0
        o = out.cpu().numpy().reshape(14, 1536, 4)
        nonzero = [bool(np.any(o[b, :, :3] != 0.0)) for b in range(14)]
        assert nonzero == [True] * 7 + [False] * 7


def test_sharded_stepper_symmetric_mode_world1_and_two_emulated_ranks():
    """ShardedStepper in symmetric mode through the C ABI at world size 1 (10 steps of config 1 against the oracle,
    tracer rows bit-exact), and one step of a 2-rank run emulated on this GPU: both ranks' shares of the pairs summed
    (the all-reduce), then each rank's kick-drift of its own slice -- equal to the world-size-1 step to rounding."""
    import torch
    from paper_1208_3444_b200.harness import Session
    from paper_1208_3444_b200.sharded import LibcolatusOps, ShardedStepper
    cfg, pm, vel = inputs.make_config(1)
    steps = 10
    tr = np.arange(0, cfg.n, cfg.n // 16, dtype=np.int32)
    mids, _ = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, steps)
    with Session(cfg.G, cfg.n) as s:
        pos, v = s.to_device(pm), s.to_device(vel)
        ops = LibcolatusOps(pos, v, torch.zeros_like(pos), cfg.n, cfg.eps2, 0, cfg.n)
        stepper = ShardedStepper(pos, cfg.n, ops, symmetric=True)
        assert stepper.symmetric and stepper.acc_full.shape == pos.shape
        idx = torch.from_numpy(tr).to(pos.device)
        ring = torch.zeros((steps, tr.size, 4), dtype=torch.float32, device=pos.device)
        ops.trace(idx, ring, steps)
        for a, H in mids:
            stepper.step(cfg.tau, a, H)
        rows = stepper.trace_read(tr, 0, steps)
        torch.cuda.synchronize()
        x_gpu, v_gpu = pos.cpu().numpy(), v.cpu().numpy()
        assert stepper.reduces == 0 and stepper.gathers == 0
    st = oracle.State(pm, vel, cfg.eps2, cfg.G)
    for a, H in mids:
        st.step(cfg.tau, a, H)
    assert np.linalg.norm(x_gpu[:, :3].astype(np.float64) - st.x, axis=1).max() <= 1e-5          # G16
    assert np.array_equal(rows[-1, :, :3], v_gpu[tr, :3])

    c = B.colatus_step_coefficients(cfg.tau, 0.05, 3.0)
    half = cfg.n // 2
    rng = np.random.Generator(np.random.PCG64(5))
    vel2 = vel.copy()
    vel2[:, :3] = 0.05 * rng.standard_normal((cfg.n, 3)).astype(np.float32)
    with Session(cfg.G, cfg.n) as s:
        pos, v = s.to_device(pm), s.to_device(vel2)
        one = ShardedStepper(pos, cfg.n, LibcolatusOps(pos, v, torch.zeros_like(pos), cfg.n, cfg.eps2, 0, cfg.n),
                             symmetric=True)
        one.step_coeffs(*c)
        torch.cuda.synchronize()
        x_ref, v_ref = pos.cpu().numpy(), v.cpu().numpy()
        # two ranks: drift both slices, "all-gather", both shares of the pairs, "all-reduce", kick-drift per slice
        pos, v = s.to_device(pm), s.to_device(vel2)
        acc = torch.zeros((half, 4), dtype=torch.float32, device=pos.device)
        B.colatus_upload(pos, v, acc, cfg.n, cfg.eps2)
        for b in (0, half):
            B.colatus_set_target_range(b, half)
            B.colatus_drift(c[0])
        parts = [torch.empty_like(pos) for _ in range(2)]
        for r in range(2):
            B.colatus_forces_symmetric_part(pos, cfg.n, cfg.eps2, r, 2, parts[r])
        total = parts[0] + parts[1]
        for b in (0, half):
            B.colatus_set_target_range(b, half)
            B.colatus_kick_drift(total[b:b + half], c[1], c[2], c[3])
        torch.cuda.synchronize()
        x2, v2 = pos.cpu().numpy(), v.cpu().numpy()
    vr = float(np.sqrt((v_ref[:, :3].astype(np.float64) ** 2).sum(1).mean()))
    assert np.abs(v2[:, :3] - v_ref[:, :3]).max() <= 2e-5 * vr and np.abs(x2[:, :3] - x_ref[:, :3]).max() <= 1e-6
    assert not np.array_equal(x2[:, :3], pm[:, :3])


def test_symmetric_sharded_step_keeps_the_external_terms():
    """a share of a symmetric evaluation carries no eq. (10) source / background term (
    they would be counted once per share), so the driver adds them ONCE after the all-reduce (colatus_add_external).
    ShardedStepper in symmetric mode with both terms on must follow colatus_step -- which applies them inside the
    library -- to rounding, at world size 1 and with two ranks emulated one after the other; and must differ from the
    run without the terms (non-vacuous)."""
    import torch
    from paper_1208_3444_b200.harness import Session
    from paper_1208_3444_b200.sharded import LibcolatusOps, ShardedStepper
    cfg, pm, vel = inputs.make_config(1)
    xpsi, S = np.array([0.5, 0.5, 1.5]), 0.5
    cen, rho = np.array([0.5, 0.5, 0.5]), 1.0
    steps = 10
    mids, _ = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, steps)
    half = cfg.n // 2
    with Session(cfg.G, cfg.n) as s:
        def single(with_terms):
            if with_terms:
                B.colatus_set_deformation(xpsi, S)
                B.colatus_set_background(cen, rho)
            s.upload(pm, vel, cfg.eps2)
            for a, H in mids:
                B.colatus_step(cfg.tau, a, H)
            out = s.download()
            B.colatus_set_deformation(None, 0.0)
            B.colatus_set_background(None, 0.0)
            return out
        x_ref, v_ref = single(True)
        x_off, v_off = single(False)

        B.colatus_set_deformation(xpsi, S)
        B.colatus_set_background(cen, rho)
        pos, v = s.to_device(pm), s.to_device(vel)
        stepper = ShardedStepper(pos, cfg.n, LibcolatusOps(pos, v, torch.zeros_like(pos), cfg.n, cfg.eps2, 0, cfg.n),
                                 symmetric=True)
        for a, H in mids:
            stepper.step(cfg.tau, a, H)
        torch.cuda.synchronize()
        x1, v1 = pos.cpu().numpy(), v.cpu().numpy()

        # two ranks, one after the other: shares summed (the all-reduce), external terms once per slice, kick-drift
        pos, v = s.to_device(pm), s.to_device(vel)
        B.colatus_upload(pos, v, torch.zeros((half, 4), dtype=torch.float32, device=pos.device), cfg.n, cfg.eps2)
        for a, H in mids:
            c = B.colatus_step_coefficients(cfg.tau, a, H)
            for b in (0, half):
                B.colatus_set_target_range(b, half)
                B.colatus_drift(c[0])
            parts = [torch.empty_like(pos) for _ in range(2)]
            for r in range(2):
                B.colatus_forces_symmetric_part(pos, cfg.n, cfg.eps2, r, 2, parts[r])
            total = parts[0] + parts[1]
            for b in (0, half):
                B.colatus_set_target_range(b, half)
                B.colatus_add_external(total[b:b + half])
                B.colatus_kick_drift(total[b:b + half], c[1], c[2], c[3])
        torch.cuda.synchronize()
        x2, v2 = pos.cpu().numpy(), v.cpu().numpy()
        B.colatus_set_deformation(None, 0.0)
        B.colatus_set_background(None, 0.0)
        # with both terms off nothing is launched and the forces stay as given
        B.colatus_set_target_range(0, half)
        before = B.colatus_launch_count()
        B.colatus_add_external(total[:half])
        assert B.colatus_launch_count() == before
    vr = float(np.sqrt((v_ref[:, :3].astype(np.float64) ** 2).sum(1).mean()))
    for xs, vs in ((x1, v1), (x2, v2)):
        assert np.abs(vs[:, :3] - v_ref[:, :3]).max() <= 2e-4 * vr and np.abs(xs[:, :3] - x_ref[:, :3]).max() <= 5e-6
    assert np.abs(x_off[:, :3] - x_ref[:, :3]).max() >= 1e-3              # the terms matter in this set-up
    # and against the oracle with the same terms (readings G21 / G22; G16 bar of the 10-step trajectories)
    st = oracle.State(pm, vel, cfg.eps2, cfg.G)
    st.deformation, st.background = (xpsi, S), (cen, rho)
    for a, H in mids:
        st.step(cfg.tau, a, H)
    for xs in (x1, x2):
        assert np.linalg.norm(xs[:, :3].astype(np.float64) - st.x, axis=1).max() <= 1e-5
