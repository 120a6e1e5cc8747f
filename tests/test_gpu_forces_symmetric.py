"""The symmetric force kernel (every pair once, Newton's third law; force_sym_kernels.cuh, colatus_force_plan)
against the FP64 oracle, through the C ABI.  It is picked automatically for whole-range evaluations of at least
20480 bodies (configs 2-5: covered at full size in test_gpu_forces.py); here it is forced on at small and ragged
sizes so that every structural case is hit: 1 block (diagonal only), 2 blocks (antipodal only), odd and even
block counts, ragged last blocks, every split count, equal and general masses, chunked evaluations.
Tolerances: north_star's (G17), as in test_gpu_forces.py."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_1208_3444_b200 import binding as B  # noqa: E402
from paper_1208_3444_b200 import inputs  # noqa: E402
from conftest import record_parity  # noqa: E402
from test_gpu_forces import MAX_TOL, MEDIAN_TOL, force_errors  # noqa: E402


@pytest.fixture(scope="module")
def session():
    from paper_1208_3444_b200.harness import Session
    s = Session(1.0, 1 << 18)
    yield s
    s.close()


@pytest.fixture()
def symmetric_always():
    B.colatus_set_option("symmetric", 2)
    yield
    B.colatus_set_option("symmetric", 1)
    B.colatus_set_option("symmetric_rows", 0)
    B.colatus_set_option("symmetric_block", 0)
    B.colatus_set_option("source_splits", 0)


def _problem(n, equal_mass, seed=0):
    rng = np.random.Generator(np.random.PCG64(9100 + seed))
    pm = np.empty((n, 4), dtype=np.float32)
    half = n // 2
    pm[:half, :3] = rng.random((half, 3))
    pm[half:, :3] = 0.5 + 0.03 * rng.standard_normal((n - half, 3))          # a clump: close pairs
    pm[:, 3] = 1.0 / n if equal_mass else np.exp(0.5 * rng.standard_normal(n)) / n
    return pm[rng.permutation(n)]


@pytest.mark.parametrize("equal_mass", [False, True])
@pytest.mark.parametrize("block", [1536, 1024, 4096])
@pytest.mark.parametrize("n", [1, 2, 3, 1023, 1025, 1535, 1536, 1537, 3072, 3073, 4097, 4609, 6145, 7000, 10753, 12289, 20481])
def test_symmetric_kernel_ragged_sizes(session, symmetric_always, n, block, equal_mass):
    """All three kernel variants (blocks of 1536 bodies = 6 targets per thread, 1024 = 4 targets per thread with
    256-source tiles, 4096 = 16 targets per thread and one CTA per SM) with 1 block (diagonal only), 2 (antipodal
    only), 3, 4, 5, ... 21: odd and even counts, full and ragged last blocks; all targets against the oracle."""
    pm = _problem(n, equal_mass, seed=n)
    eps2 = np.float32(1e-4)
    B.colatus_set_option("symmetric_block", block)
    plan = B.colatus_force_plan(n)
    assert plan["symmetric"] == 1 and plan["blocks"] == (n + block - 1) // block
    assert B.colatus_force_geometry(n)["targets_per_cta"] == block
    assert plan["distances"] == (plan["blocks"] - 1) // 2
    out = session.forces(pm, eps2).cpu().numpy()
    assert np.all(out[:, 3] == 0.0)
    if n == 1:
        assert np.all(out == 0.0)
        return
    ref = oracle.forces(pm, eps2, 1.0)
    med, mx = force_errors(out[:, :3], ref)
    if n in (3073, 20481):
        record_parity(f"symmetric kernel n={n} block={block} equal_mass={equal_mass}", n=n, targets=n, median_rel=med,
                      max_over_rms=mx)
    assert med <= MEDIAN_TOL and mx <= MAX_TOL, (n, block, equal_mass, med, mx)


@pytest.mark.parametrize("splits", [1, 2, 3, 5, 7, 16])
def test_symmetric_kernel_split_counts(session, symmetric_always, splits):
    """Any split of a block's tile list (a split may begin or end inside a block, and may be empty)."""
    n = 13000                                                        # 9 blocks, H = 4: 15 tiles per block
    pm = _problem(n, False, seed=splits)
    eps2 = np.float32(2.5e-5)
    B.colatus_set_option("symmetric_block", 1536)
    B.colatus_set_option("source_splits", splits)
    plan = B.colatus_force_plan(n)
    assert plan["symmetric"] == 1 and plan["splits"] == splits
    out = session.forces(pm, eps2).cpu().numpy()
    ref = oracle.forces(pm, eps2, 1.0)
    med, mx = force_errors(out[:, :3], ref)
    assert med <= MEDIAN_TOL and mx <= MAX_TOL, (splits, med, mx)


def test_symmetric_kernel_chunked_evaluation(session, symmetric_always):
    """A cap on the partial rows per launch splits the block distances over several launches whose sums are
    accumulated: same forces (to rounding) as the single launch, and the oracle's."""
    n = 30000                                                        # 20 blocks, H = 9, antipodal block
    pm = _problem(n, False, seed=77)
    eps2 = np.float32(1e-5)
    B.colatus_set_option("symmetric_block", 1536)
    B.colatus_set_option("source_splits", 3)
    one = session.forces(pm, eps2).cpu().numpy()
    assert B.colatus_force_plan(n)["launches"] == 1
    ref = oracle.forces(pm, eps2, 1.0)
    for rows, launches in ((3 + 4, 3), (3 + 1, 9), (3 + 5, 2)):
        B.colatus_set_option("symmetric_rows", rows)
        plan = B.colatus_force_plan(n)
        assert plan["launches"] == launches and plan["distances_per_launch"] == rows - 3, plan
        out = session.forces(pm, eps2).cpu().numpy()
        med, mx = force_errors(out[:, :3], ref)
        assert med <= MEDIAN_TOL and mx <= MAX_TOL, (rows, med, mx)
        assert np.abs(out - one).max() <= 2e-6 * np.abs(one).max()


def test_symmetric_kernel_matches_one_directional_kernel(session, symmetric_always):
    """Same problem through both kernels: equal to FP32 summation rounding, both within the bars; the symmetric
    result obeys Newton's third law to rounding (sum m F = 0), and is bitwise reproducible."""
    cfg, pm, _ = inputs.make_config(3, n_override=40000)
    sym = session.forces(pm, cfg.eps2).cpu().numpy()
    again = session.forces(pm, cfg.eps2).cpu().numpy()
    assert np.array_equal(sym, again)
    B.colatus_set_option("symmetric", 0)
    assert B.colatus_force_plan(cfg.n)["symmetric"] == 0
    plain = session.forces(pm, cfg.eps2).cpu().numpy()
    ref = oracle.forces(pm, cfg.eps2, 1.0)
    for name, out in (("symmetric", sym), ("one-directional", plain)):
        med, mx = force_errors(out[:, :3], ref)
        record_parity(f"config-3-shaped n=40000 {name} kernel", n=cfg.n, targets=cfg.n, median_rel=med, max_over_rms=mx)
        assert med <= MEDIAN_TOL and mx <= MAX_TOL, (name, med, mx)
    m = pm[:, 3].astype(np.float64)
    F = sym[:, :3].astype(np.float64)
    assert np.linalg.norm((m[:, None] * F).sum(0)) / (m * np.linalg.norm(F, axis=1)).sum() < 2e-6


def test_symmetric_kernel_masses(session, symmetric_always):
    """Equal-mass detection inside the symmetric kernel: one different mass (also 0) is honoured; all-zero masses
    give exact zeros; a NaN mass gives NaN forces, not an error."""
    n = 5000
    pm0 = _problem(n, True, seed=5)
    eps2 = np.float32(1e-4)
    for where, factor in ((0, 3.0), (2500, 0.0), (4999, 50.0)):
        pm = pm0.copy()
        pm[where, 3] *= factor
        out = session.forces(pm, eps2).cpu().numpy()
        ref = oracle.forces(pm, eps2, 1.0)
        med, mx = force_errors(out[:, :3], ref)
        assert med <= MEDIAN_TOL and mx <= MAX_TOL, (where, factor, med, mx)
    z = pm0.copy()
    z[:, 3] = 0.0
    assert np.all(session.forces(z, eps2).cpu().numpy() == 0.0)
    q = pm0.copy()
    q[7, 3] = np.nan
    out = session.forces(q, eps2).cpu().numpy()
    assert np.isnan(out[:, :3]).all(axis=1).sum() >= n - 1


def test_symmetric_kernel_at_the_smallest_accepted_eps2(session, symmetric_always):
    """Coincident bodies and the eps2 floor (reading G4): the pair term of coincident bodies is exactly 0 in both
    directions."""
    n = 4000
    pm = _problem(n, False, seed=11)
    pm[100, :3] = pm[3000, :3]                                       # two coincident bodies in different blocks
    pm[200, :3] = pm[201, :3]                                        # ... and in the same block
    eps2 = np.float32(1e-24)
    out = session.forces(pm, eps2).cpu().numpy()
    assert np.isfinite(out).all()
    ref = oracle.forces(pm, eps2, 1.0)
    med, mx = force_errors(out[:, :3], ref)
    assert med <= MEDIAN_TOL and mx <= MAX_TOL, (med, mx)


def test_symmetric_steps_match_the_oracle_and_the_run_loop(session, symmetric_always):
    """10 steps of config 1 with the symmetric kernel inside colatus_step (fused kick) and inside colatus_run
    (two-kernel loop, graphs): the 10-step bar against the oracle (G16), and run == step loop bit for bit."""
    cfg, pm, vel = inputs.make_config(1)
    assert cfg.G == 1.0
    s = session
    if True:
        assert B.colatus_force_plan(cfg.n)["symmetric"] == 1
        steps = 10
        mids, _ = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, steps)
        s.upload(pm, vel, cfg.eps2)
        s.run(cfg.cosmo, cfg.a_start, cfg.tau, steps)
        pos_a, vel_a = s.download()
        st = oracle.State(pm, vel, cfg.eps2, cfg.G)
        for a, H in mids:
            st.step(cfg.tau, a, H)
        dx = float(np.linalg.norm(pos_a[:, :3].astype(np.float64) - st.x, axis=1).max())
        assert dx <= 1e-5, dx
        for use_graph in (False, True):
            s.upload(pm, vel, cfg.eps2)
            s.run_native(cfg.cosmo, cfg.a_start, cfg.tau, steps, use_graph=use_graph)
            pos_b, vel_b = s.download()
            assert np.array_equal(pos_a, pos_b) and np.array_equal(vel_a, vel_b), use_graph


def test_symmetric_chunked_steps(session, symmetric_always):
    """Steps whose force evaluation takes several launches of the symmetric kernel (partial rows capped): the kick
    reads the accumulated forces; colatus_run (graphs, plain launches) == colatus_step loop bit for bit, and the
    trajectory agrees with the single-launch one to rounding."""
    n = 13000                                                        # 9 blocks, H = 4
    pm = _problem(n, True, seed=3)
    vel = np.zeros_like(pm)
    eps2 = np.float32(1e-4)
    steps, tau = 5, 1e-3
    s = session
    results = {}
    for rows in (0, 6):                                              # automatic (1 launch) / 4 + 2 rows (2 launches)
        B.colatus_set_option("symmetric_block", 1536)
        B.colatus_set_option("source_splits", 4)
        B.colatus_set_option("symmetric_rows", rows)
        assert B.colatus_force_plan(n)["launches"] == (1 if rows == 0 else 2)
        s.upload(pm, vel, eps2)
        s.trace(np.arange(0, n, n // 16, dtype=np.int32)[:16], steps)
        s.run(None, 1.0, tau, steps)
        pos_a, vel_a = s.download()
        tr_a = s.trace_read(0, steps)
        for use_graph in (False, True):
            s.upload(pm, vel, eps2)
            s.trace(np.arange(0, n, n // 16, dtype=np.int32)[:16], steps)
            s.run_native(None, 1.0, tau, steps, use_graph=use_graph)
            pos_b, vel_b = s.download()
            assert np.array_equal(pos_a, pos_b) and np.array_equal(vel_a, vel_b), (rows, use_graph)
            assert np.array_equal(tr_a, s.trace_read(0, steps))
        results[rows] = (pos_a, vel_a)
    assert np.abs(results[0][0][:, :3] - results[6][0][:, :3]).max() < 1e-6
    st = oracle.State(pm, vel, eps2, 1.0)
    for _ in range(steps):
        st.step(tau, 1.0, 0.0)
    assert float(np.linalg.norm(results[6][0][:, :3].astype(np.float64) - st.x, axis=1).max()) <= 1e-5


def test_plan_of_the_baseline_configurations(session):
    """What colatus_force_plan reports for BASELINE.json's sizes on this device."""
    if True:
        small = B.colatus_force_plan(4096)
        assert small["symmetric"] == 0
        for n in (32768, 100000, 131072, 262144):                                # all rows fit the 512 MiB budget
            p = B.colatus_force_plan(n)
            block = 1024 if n < 65536 else 4096
            assert p["symmetric"] == 1 and p["launches"] == 1 and p["blocks"] == (n + block - 1) // block
            assert p["partial_rows"] == p["splits"] + p["distances"]
        for n, row_bytes in ((1 << 20, 512 << 20), (1 << 22, 2 << 30)):          # beyond it: 32 rows per launch
            big = B.colatus_force_plan(n)
            assert big["symmetric"] == 1 and big["launches"] > 1 and big["partial_rows"] == 32
            assert big["partial_rows"] == big["splits"] + big["distances_per_launch"]
            assert big["partial_rows"] * big["padded_bodies"] * 16 == row_bytes
        assert B.colatus_force_plan(1 << 20, 1 << 19)["symmetric"] == 0          # target sub-range
        pot = B.colatus_force_plan(1 << 20, None, True)                          # potential: 1024-body blocks, chunked
        assert pot["symmetric"] == 1 and pot["blocks"] == 1024 and pot["launches"] > 1
        assert pot["partial_rows"] * pot["padded_bodies"] * 16 <= 512 << 20


@pytest.mark.parametrize("seed", range(16))
def test_symmetric_kernel_fuzz_against_the_one_directional_kernel(session, symmetric_always, seed):
    """Seeded random problem sizes (2 .. 70000: 1 to 69 blocks, odd and even), block sizes, split counts and row caps
    (1 to ~20 launches), equal and general masses, scales and offsets: the symmetric evaluation agrees with the
    one-directional kernel -- which test_gpu_forces.py holds to the oracle at every size -- far inside the bars, and
    with the oracle itself where it is cheap (n <= 20000)."""
    rng = np.random.Generator(np.random.PCG64(4400 + seed))
    n = int(rng.integers(2, 70000)) if seed % 4 else int(rng.integers(2, 5000))
    block = (0, 1024, 1536, 4096)[int(rng.integers(0, 4))]
    splits = int(rng.integers(0, 17))
    scale = 10.0 ** rng.uniform(-2, 2)
    pm = _problem(n, bool(seed % 2), seed=seed)
    pm[:, :3] = (scale * (pm[:, :3] + rng.uniform(-20, 20, size=3))).astype(np.float32)
    eps2 = np.float32((scale * 10.0 ** rng.uniform(-3, -1.5)) ** 2)
    B.colatus_set_option("symmetric_block", block)
    B.colatus_set_option("source_splits", splits)
    plan = B.colatus_force_plan(n)
    if plan["distances"] > 2 and seed % 3 == 0:
        B.colatus_set_option("symmetric_rows", plan["splits"] + int(rng.integers(1, plan["distances"])))
        plan = B.colatus_force_plan(n)
    assert plan["symmetric"] == 1
    sym = session.forces(pm, eps2).cpu().numpy()
    B.colatus_set_option("symmetric", 0)
    B.colatus_set_option("source_splits", 0)
    plain = session.forces(pm, eps2).cpu().numpy()
    ref = plain[:, :3].astype(np.float64)
    med, mx = force_errors(sym[:, :3], ref)
    assert med <= 2e-6 and mx <= 2e-5, (seed, n, block, splits, plan, med, mx)
    if n <= 20000:
        med, mx = force_errors(sym[:, :3], oracle.forces(pm, eps2, 1.0))
        assert med <= MEDIAN_TOL and mx <= MAX_TOL, (seed, n, med, mx)


@pytest.mark.parametrize("equal_mass", [False, True])
@pytest.mark.parametrize("n", [1, 2, 1025, 3073, 30000])
def test_symmetric_kernel_with_the_potential(session, symmetric_always, n, equal_mass):
    """colatus_forces_potential through the symmetric kernel (fourth component: the potential is symmetric in the
    pair, the j = k term of the diagonal tiles is removed by the row reduction): forces and phi against the oracle,
    one launch and chunked over block distances."""
    pm = _problem(n, equal_mass, seed=100 + n)
    eps2 = np.float32(1e-4)
    plan = B.colatus_force_plan(n, None, True)
    assert plan["symmetric"] == 1 and plan["blocks"] == (n + 1023) // 1024
    ref, phi = oracle.forces(pm, eps2, 1.0, potential=True)
    for rows in ((0, 5) if n == 30000 else (0,)):
        B.colatus_set_option("symmetric_rows", rows)
        if rows:
            B.colatus_set_option("source_splits", 2)
            assert B.colatus_force_plan(n, None, True)["launches"] == 5          # H = 14, 3 distances per launch
        out = session.forces(pm, eps2, potential=True).cpu().numpy()
        if n == 1:       # phi = -(m / eps - m / eps): the removed j = k term leaves at most its own rounding
            assert np.all(out[:, :3] == 0.0) and abs(out[0, 3]) <= 2e-7 * pm[0, 3] / np.sqrt(eps2)
            continue
        med, mx = force_errors(out[:, :3], ref)
        assert med <= MEDIAN_TOL and mx <= MAX_TOL, (n, equal_mass, rows, med, mx)
        assert np.allclose(out[:, 3], phi, rtol=5e-5, atol=0), (n, equal_mass, rows)
