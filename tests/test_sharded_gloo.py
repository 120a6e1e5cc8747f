"""World-size-2 CPU test (gloo) of the target-sharded multi-GPU sequencing (DESIGN.md "Multi-GPU",
SURVEY 8e): ShardedStepper must drift / force-kick-drift only its own slice, all-gather positions
ONCE per step (after the first drift; lazily before a read of full positions), reduce the diagnostics
with one all-reduce, assemble the tracer rows from the owning ranks, and reproduce the single-process
trajectory exactly.

No GPU here, so the per-slice work is done by a stand-in `ops` built on the FP64 oracle (tests may
use the oracle); what is under test is the host-side sequencing and the exchange step in
`paper_1208_3444_b200/sharded.py`, which is the same code the NCCL path runs.
"""
from __future__ import annotations

import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_1208_3444_b200 import inputs
from paper_1208_3444_b200.sharded import ShardedStepper, partition

N, STEPS, WORLD = 512, 4, 2


TRACERS = np.array([3, 100, 255, 256, 400, 511], dtype=np.int64)     # both slices, including their edges


class OracleSliceOps:
    """Drift / force+kick+drift of eqs. (3)-(5) on the slice [begin, begin+count) of float64 state, the
    slice diagnostics in colatus_diagnostics' layout, and a tracer ring that (like libcolatus with a target
    range) records only the tracers this rank owns.

    `pos` is the [n,4] float64 tensor ShardedStepper all-gathers; velocities exist for the slice only."""

    def __init__(self, pos, vel_slice, eps2, G, begin, count, steps):
        self.pos, self.vel, self.eps2, self.G = pos, vel_slice, eps2, G
        self.begin, self.count = begin, count
        self.step = 0
        self.ring = np.zeros((steps, TRACERS.size, 4), dtype=np.float32)

    def drift(self, d):
        s = slice(self.begin, self.begin + self.count)
        self.pos[s, :3] += d * self.vel

    def force_kick_drift(self, cv, ck, d2):
        x = self.pos[:, :3].numpy()
        m = self.pos[:, 3].numpy()
        targets = np.arange(self.begin, self.begin + self.count, dtype=np.int64)
        F = torch.from_numpy(oracle.forces_xm(x, m, self.eps2, self.G, targets))
        self.vel.mul_(cv).add_(ck * F)
        s = slice(self.begin, self.begin + self.count)
        self.pos[s, :3] += d2 * self.vel
        for t, k in enumerate(TRACERS):
            if self.begin <= k < self.begin + self.count:
                self.ring[self.step, t, :3] = self.vel[k - self.begin].numpy()
                self.ring[self.step, t, 3] = 1.0
        self.step += 1

    def diagnostics(self, a, with_potential=False):
        s = slice(self.begin, self.begin + self.count)
        x, m, v = self.pos[s, :3].numpy(), self.pos[s, 3].numpy(), self.vel.numpy()
        out = np.zeros(16)
        out[0] = m.sum()
        out[1:4] = (m[:, None] * v).sum(0)
        out[4:7] = a * a * out[1:4]
        out[7] = 0.5 * a * a * (m * (v * v).sum(1)).sum()
        out[8] = np.nan
        if with_potential:
            targets = np.arange(self.begin, self.begin + self.count, dtype=np.int64)
            _, phi = oracle.forces_xm(self.pos[:, :3].numpy(), self.pos[:, 3].numpy(), self.eps2, self.G, targets, True)
            out[8] = 0.5 * (m * phi).sum() / a
        out[13:16] = (m[:, None] * x).sum(0)
        out[9:12] = out[13:16] / out[0]
        out[12] = self.step
        return out

    def trace_rows(self, first_step, n_steps):
        return self.ring[first_step:first_step + n_steps].copy()

    # ---- symmetric mode: this rank's share of the unordered pairs, on ALL bodies; then the kick from given forces
    BLOCK = 32                       # bodies per block of the stand-in's circulant pairing

    def forces_symmetric_part(self, part, parts, acc_full):
        """Same division of the work as colatus_forces_symmetric_part (target blocks [nb part / parts, nb (part+1) /
        parts); block a meets a+1 .. a+H both ways, itself and -- nb even -- the antipodal block one way), in FP64
        with numpy: the pair term is computed ONCE and added to both bodies."""
        x, m = self.pos[:, :3].numpy(), self.pos[:, 3].numpy()
        n, B_ = x.shape[0], self.BLOCK
        nb = (n + B_ - 1) // B_
        H = (nb - 1) // 2
        F = np.zeros((n, 3))
        blk = lambda b: np.arange(b * B_, min((b + 1) * B_, n))

        def one_way(ti, sj):
            d = x[sj][None, :, :] - x[ti][:, None, :]
            s2 = (d * d).sum(2) + self.eps2
            w = m[sj][None, :] / (s2 * np.sqrt(s2))
            w[ti[:, None] == sj[None, :]] = 0.0
            F[ti] += self.G * (w[:, :, None] * d).sum(1)

        for a in range(nb * part // parts, nb * (part + 1) // parts):
            ti = blk(a)
            one_way(ti, ti)
            if nb % 2 == 0 and nb > 1:
                one_way(ti, blk((a + nb // 2) % nb))
            for k in range(1, H + 1):
                sj = blk((a + k) % nb)
                d = x[sj][None, :, :] - x[ti][:, None, :]
                s2 = (d * d).sum(2) + self.eps2
                g = d / (s2 * np.sqrt(s2))[:, :, None]                     # the antisymmetric pair term, once
                F[ti] += self.G * (m[sj][None, :, None] * g).sum(1)        # action
                F[sj] -= self.G * (m[ti][:, None, None] * g).sum(0)        # reaction
        acc_full[:, :3] = torch.from_numpy(F)
        acc_full[:, 3] = 0.0

    external_calls = 0

    def add_external(self, acc_slice):
        """Stand-in for colatus_add_external: once per step, on the summed forces of the own slice."""
        self.external_calls += 1

    def kick_drift(self, acc_slice, cv, ck, d2):
        self.vel.mul_(cv).add_(ck * acc_slice[:, :3])
        s = slice(self.begin, self.begin + self.count)
        self.pos[s, :3] += d2 * self.vel
        for t, k in enumerate(TRACERS):
            if self.begin <= k < self.begin + self.count:
                self.ring[self.step, t, :3] = self.vel[k - self.begin].numpy()
                self.ring[self.step, t, 3] = 1.0
        self.step += 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, pm, vel, eps2, G, coeffs, out_dir, symmetric=False):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        pos = torch.from_numpy(pm.astype(np.float64))
        begin, count = partition(pm.shape[0], world, rank)
        v = torch.from_numpy(vel[begin:begin + count, :3].astype(np.float64))
        stepper = ShardedStepper(pos, pm.shape[0], OracleSliceOps(pos, v, eps2, G, begin, count, len(coeffs)),
                                 symmetric=symmetric)
        assert (stepper.begin, stepper.count) == (begin, count) and stepper.symmetric == symmetric
        for c in coeffs:
            stepper.step_coeffs(*c)
        assert stepper.gathers == len(coeffs) and stepper.dirty          # ONE all-gather per step
        assert stepper.reduces == (len(coeffs) if symmetric else 0)       # symmetric mode: + ONE all-reduce of forces
        assert stepper.ops.external_calls == (len(coeffs) if symmetric else 0)   # external terms: once, after the sum
        other = slice(0, count) if rank == 1 else slice(count, 2 * count)
        stale = pos[other].clone()
        d_kin = stepper.diagnostics(0.5)                                  # no potential: no gather needed
        assert stepper.gathers == len(coeffs) and torch.equal(pos[other], stale)
        d_pot = stepper.diagnostics(0.5, with_potential=True)             # W reads all sources: lazy gather
        assert stepper.gathers == len(coeffs) + 1 and not stepper.dirty and not torch.equal(pos[other], stale)
        stepper.sync_positions()
        assert stepper.gathers == len(coeffs) + 1                         # already current
        rows = stepper.trace_read(TRACERS, 0, len(coeffs))
        np.save(os.path.join(out_dir, f"pos{rank}.npy"), pos.numpy())
        np.save(os.path.join(out_dir, f"vel{rank}.npy"), v.numpy())
        np.save(os.path.join(out_dir, f"diag{rank}.npy"), np.stack([d_kin, d_pot]))
        np.save(os.path.join(out_dir, f"rows{rank}.npy"), rows)
    finally:
        dist.destroy_process_group()


def test_partition():
    assert partition(1024, 4, 0) == (0, 256) and partition(1024, 4, 3) == (768, 256)
    with pytest.raises(ValueError):
        partition(1000, 3, 0)


@pytest.mark.parametrize("symmetric", [False, True])
def test_two_rank_sharded_stepping_matches_single_process(tmp_path, symmetric):
    """symmetric=False: eq. (1) divided by targets; True: by block pairs, every pair evaluated once by one of the two
    ranks, action and reaction delivered by one all-reduce of the partial forces (sharded.py)."""
    cfg, pm, vel = inputs.make_config(1, n_override=N)
    rng = np.random.Generator(np.random.PCG64(7))
    vel = vel.copy()
    vel[:, :3] = 0.05 * rng.standard_normal((N, 3)).astype(np.float32)
    mids, _ = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, STEPS)
    coeffs = []
    for a, H in mids:          # eqs. (3)-(5): d1, cv, ck, d2
        coeffs.append((0.5 * cfg.tau, (1 - H * cfg.tau) / (1 + H * cfg.tau),
                       cfg.tau / (a ** 3 * (1 + H * cfg.tau)), 0.5 * cfg.tau))

    mp.spawn(_worker, args=(WORLD, _free_port(), pm, vel, float(cfg.eps2), cfg.G, coeffs, str(tmp_path), symmetric),
             nprocs=WORLD, join=True)

    ref = oracle.State(pm, vel, cfg.eps2, cfg.G)
    rows_ref = np.zeros((STEPS, TRACERS.size, 4), dtype=np.float32)
    for n, c in enumerate(coeffs):
        ref.step_coeffs(*c)
        rows_ref[n, :, :3] = ref.v[TRACERS]
        rows_ref[n, :, 3] = 1.0
    pos0 = np.load(tmp_path / "pos0.npy")
    pos1 = np.load(tmp_path / "pos1.npy")
    assert np.array_equal(pos0, pos1)                      # every rank ends with the same full position array
    # target sharding: same arithmetic, per-target sums in the same order; pair sharding: another summation order (FP64)
    assert np.abs(pos0[:, :3] - ref.x).max() <= (1e-12 if symmetric else 1e-14)
    v = np.concatenate([np.load(tmp_path / "vel0.npy"), np.load(tmp_path / "vel1.npy")])
    assert np.abs(v - ref.v).max() <= (1e-10 if symmetric else 1e-13)
    assert np.array_equal(pos0[:, 3], pm[:, 3].astype(np.float64))   # masses untouched by the exchange

    # diagnostics: one all-reduce of the 16 doubles gives the whole-system sums on every rank
    d0, d1 = np.load(tmp_path / "diag0.npy"), np.load(tmp_path / "diag1.npy")
    assert np.array_equal(d0[1], d1[1]) and np.array_equal(d0[0, :8], d1[0, :8])
    dref = ref.diagnostics(0.5, with_potential=True)
    for i in range(0, 12):
        assert d0[1][i] == pytest.approx(dref[i], rel=1e-12, abs=1e-15), i
    assert d0[1][13:16] == pytest.approx(dref[9:12] * dref[0], rel=1e-12)       # sum m x (additive over shards)
    assert np.isnan(d0[0][8]) and d0[0][7] == pytest.approx(dref[7], rel=1e-12)
    assert d0[1][12] == STEPS
    # tracers: each row comes from the rank that owns the particle; both ranks assemble the same full record
    r0, r1 = np.load(tmp_path / "rows0.npy"), np.load(tmp_path / "rows1.npy")
    assert np.array_equal(r0, r1)
    assert np.array_equal(r0[:, :, 3], rows_ref[:, :, 3]) and np.abs(r0[:, :, :3] - rows_ref[:, :, :3]).max() <= 1e-7 * np.abs(rows_ref).max()
