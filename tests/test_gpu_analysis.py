"""GPU parity for NEXT rows f4 (headless particle-count snapshot; Fig. 1 PAPER.md:83-85;
reading G23) and f3 (tracer velocity power spectrum; reading G24) against the oracle,
through the C ABI.  The image is integer work: bit-exact.  The spectrum is FP64 on both sides from the
same FP32 samples: 1e-10 of the record's largest bin."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_1208_3444_b200 import binding as B  # noqa: E402
from paper_1208_3444_b200 import inputs  # noqa: E402

SPECTRUM_RTOL = 1e-10


def _session(G, n):
    from paper_1208_3444_b200.harness import Session
    return Session(G, n)


WINDOWS = [
    (2, (0.0, 1.0, 0.0, 1.0, -np.inf, np.inf), 256, 256),        # whole box, as Fig. 1
    (0, (0.1, 0.9, 0.2, 0.7, 0.25, 0.5), 37, 23),                # ragged image, slab, non-dyadic scale
    (1, (0.4, 0.6, 0.4, 0.6, 0.45, 0.55), 1024, 512),            # zoom on a dense region
    (2, (-1.0, 2.0, -1.0, 2.0, 0.0, 1.0), 3, 1),                 # coarse, window larger than the box
]


@pytest.mark.parametrize("index", [2, 3, 4])
def test_splat_matches_oracle_bit_exact(index):
    cfg, pm, _ = inputs.make_config(index)
    with _session(cfg.G, cfg.n) as s:
        dev = s.to_device(pm)
        for axis, win, W, H in WINDOWS:
            got = s.splat(axis, win, W, H, pos_mass=dev)
            want = oracle.splat(pm, axis, win, W, H)
            assert got.shape == (H, W) and got.dtype == np.uint32
            assert np.array_equal(got, want), (index, axis, win)
            assert want.sum() > 0
    # whole box, no slab: every particle with (x, y) inside [0,1)^2 is counted once
    inside = np.all((pm[:, :2] >= 0) & (pm[:, :2] < 1), axis=1).sum()
    assert oracle.splat(pm, 2, WINDOWS[0][1], 256, 256).sum() == inside


def test_splat_edge_cases():
    """n = 1, a clump of coincident particles (warp-merged atomics), particles exactly on the window edges,
    NaN positions, and a buffer that is re-zeroed by every call."""
    pm = np.zeros((1000, 4), dtype=np.float32)
    pm[:, :3] = 0.5                                   # 1000 coincident bodies -> one pixel
    pm[0, :3] = (0.0, 0.0, 0.0)                       # lower edge: inside
    pm[1, :3] = (1.0, 0.5, 0.5)                       # upper edge in u: outside
    pm[2, :3] = (np.nan, 0.5, 0.5)
    pm[3, :3] = (0.5, np.inf, 0.5)
    win = (0.0, 1.0, 0.0, 1.0, 0.0, 1.0)
    with _session(1.0, 1000) as s:
        for _ in range(2):
            got = s.splat(2, win, 8, 8, pos_mass=pm)
            assert np.array_equal(got, oracle.splat(pm, 2, win, 8, 8))
        assert got[4, 4] == 996 and got[0, 0] == 1 and got.sum() == 997
        one = s.splat(2, win, 5, 7, pos_mass=pm[:1])
        assert one.sum() == 1 and one[0, 0] == 1


def test_splat_of_resident_state_after_steps():
    """pos_mass_dev = NULL images the resident positions: identical to imaging the downloaded array."""
    cfg, pm, vel = inputs.make_config(1)
    rng = np.random.Generator(np.random.PCG64(77))
    vel = vel.copy()
    vel[:, :3] = 5.0 * rng.standard_normal((cfg.n, 3)).astype(np.float32)
    win = (0.0, 1.0, 0.0, 1.0, -np.inf, np.inf)
    with _session(cfg.G, cfg.n) as s:
        s.upload(pm, vel, cfg.eps2)
        before = s.splat(2, win, 64, 64)
        assert np.array_equal(before, oracle.splat(pm, 2, win, 64, 64))
        s.run(cfg.cosmo, cfg.a_start, cfg.tau, 3)
        after = s.splat(2, win, 64, 64)
        pos, _ = s.download()
        again = s.splat(2, win, 64, 64, pos_mass=pos)
    assert np.array_equal(after, again)
    assert not np.array_equal(before, after)


def test_splat_argument_validation():
    cfg, pm, _ = inputs.make_config(1)
    with _session(1.0, cfg.n) as s:
        import torch
        dev = s.to_device(pm)
        img = torch.zeros((4, 4), dtype=torch.int32, device=s.device)
        ok = (0.0, 1.0, 0.0, 1.0, 0.0, 1.0)
        for bad in ((1.0, 1.0, 0.0, 1.0, 0.0, 1.0), (0.0, 1.0, 1.0, 0.0, 0.0, 1.0), (0.0, 1.0, 0.0, 1.0, 1.0, 1.0),
                    (0.0, np.inf, 0.0, 1.0, 0.0, 1.0), (np.nan, 1.0, 0.0, 1.0, 0.0, 1.0)):
            with pytest.raises(B.ColatusError):
                B.colatus_splat(dev, cfg.n, 2, bad, 4, 4, img)
        for axis, W, H in ((3, 4, 4), (-1, 4, 4), (0, 0, 4), (0, 4, 40000)):
            with pytest.raises(B.ColatusError):
                B.colatus_splat(dev, cfg.n, axis, ok, W, H, img)
        with pytest.raises(B.ColatusError):
            B.colatus_splat(None, 0, 2, ok, 4, 4, img)            # no resident state
        with pytest.raises(B.ColatusError):
            B.colatus_splat(dev, cfg.n, 2, ok, 4, 4, None)


# ------------------------------------------------------------------------------------------ f3
@pytest.mark.parametrize("steps,capacity,first", [(64, 64, 0), (45, 64, 0), (50, 40, 10), (200, 256, 37)])
def test_trace_spectrum_matches_oracle(steps, capacity, first):
    """The GPU periodogram of the ring equals the oracle's periodogram of the rows read back with
    colatus_trace_read (same FP32 samples; ring wrap-around and odd S covered)."""
    cfg, pm, vel = inputs.make_config(1)
    rng = np.random.Generator(np.random.PCG64(5))
    vel = vel.copy()
    vel[:, :3] = 0.3 * rng.standard_normal((cfg.n, 3)).astype(np.float32)
    idx = np.arange(0, cfg.n, cfg.n // 48, dtype=np.int32)[:48]
    S = steps - first
    with _session(cfg.G, cfg.n) as s:
        s.upload(pm, vel, cfg.eps2)
        s.trace(idx, capacity)
        s.run(cfg.cosmo, cfg.a_start, cfg.tau, steps)
        rows = s.trace_read(first, S)
        got = s.trace_spectrum(first, S)
    want = oracle.trace_spectrum(rows)
    assert got.shape == want.shape == (48, S // 2 + 1)
    assert np.abs(got - want).max() <= SPECTRUM_RTOL * want.max()
    assert want.max() > 0 and np.count_nonzero(want > 1e-3 * want.max()) > 10      # a real spectrum
    # Parseval on the GPU result itself
    wgt = np.full(S // 2 + 1, 2.0)
    wgt[0] = 1.0
    if S % 2 == 0:
        wgt[-1] = 1.0
    energy = (rows[:, :, :3].astype(np.float64) ** 2).sum((0, 2))
    assert np.allclose((got * wgt).sum(1), energy, rtol=1e-10)


def test_trace_spectrum_of_an_orbit_peaks_at_the_orbital_frequency():
    """Two equal bodies on a softened circular orbit (static background): the velocity series of either
    is a sinusoid at the orbital frequency, so the spectrum has a single interior peak there."""
    G, m, r, eps2 = 1.0, 0.5, 0.5, 0.01
    d = 2 * r
    vc = np.sqrt(G * m * d * r / (d * d + eps2) ** 1.5)              # v^2/r = G m d/(d^2+eps^2)^{3/2}
    period = 2 * np.pi * r / vc
    S, orbits = 256, 8
    tau = orbits * period / S
    pm = np.array([[0.5 + r, 0.5, 0.5, m], [0.5 - r, 0.5, 0.5, m]], dtype=np.float32)
    vel = np.array([[0, vc, 0, 0], [0, -vc, 0, 0]], dtype=np.float32)
    with _session(G, 2) as s:
        s.upload(pm, vel, eps2)
        s.trace(np.array([0, 1], dtype=np.int32), S)
        s.run(None, 1.0, tau, S)
        got = s.trace_spectrum(0, S)
        rows = s.trace_read(0, S)
    assert np.abs(got - oracle.trace_spectrum(rows)).max() <= SPECTRUM_RTOL * got.max()
    for t in range(2):
        assert int(np.argmax(got[t])) == orbits
        assert got[t, orbits] >= 0.95 * got[t].sum()        # leapfrog phase error leaks a little
        assert got[t, orbits] == pytest.approx(S * vc * vc / 2, rel=5e-2)      # S A^2/4 per component, two components


def test_trace_spectrum_argument_validation():
    cfg, pm, vel = inputs.make_config(1)
    import torch
    with _session(cfg.G, cfg.n) as s:
        out = torch.zeros((4, 9), dtype=torch.float64, device=s.device)
        with pytest.raises(B.ColatusError):
            B.colatus_trace_spectrum(0, 16, out)                    # not uploaded
        s.upload(pm, vel, cfg.eps2)
        with pytest.raises(B.ColatusError):
            B.colatus_trace_spectrum(0, 16, out)                    # no tracers
        s.trace(np.arange(4, dtype=np.int32), 8)
        s.run(cfg.cosmo, cfg.a_start, cfg.tau, 12)
        for first, S in ((0, 8), (4, 16), (8, 1), (-1, 4), (6, 8)):
            with pytest.raises(B.ColatusError):
                B.colatus_trace_spectrum(first, S, out)
        with pytest.raises(B.ColatusError):
            B.colatus_trace_spectrum(4, 8, None)
        B.colatus_trace_spectrum(4, 8, out)                         # steps 4..11 are held
