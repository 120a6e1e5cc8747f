"""World-size-2 CPU test (gloo) of the target-sharded multi-GPU sequencing (DESIGN.md "Multi-GPU",
SURVEY 8e): ShardedStepper must drift / force-kick-drift only its own slice, all-gather positions
after every drift, and reproduce the single-process trajectory exactly.

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


class OracleSliceOps:
    """Drift / force+kick+drift of eqs. (3)-(5) on the slice [begin, begin+count) of float64 state.

    `pos` is the [n,4] float64 tensor ShardedStepper all-gathers; velocities exist for the slice only."""

    def __init__(self, pos, vel_slice, eps2, G, begin, count):
        self.pos, self.vel, self.eps2, self.G = pos, vel_slice, eps2, G
        self.begin, self.count = begin, count

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


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, pm, vel, eps2, G, coeffs, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        pos = torch.from_numpy(pm.astype(np.float64))
        begin, count = partition(pm.shape[0], world, rank)
        v = torch.from_numpy(vel[begin:begin + count, :3].astype(np.float64))
        stepper = ShardedStepper(pos, pm.shape[0], OracleSliceOps(pos, v, eps2, G, begin, count))
        assert (stepper.begin, stepper.count) == (begin, count)
        for c in coeffs:
            stepper.step_coeffs(*c)
        np.save(os.path.join(out_dir, f"pos{rank}.npy"), pos.numpy())
        np.save(os.path.join(out_dir, f"vel{rank}.npy"), v.numpy())
    finally:
        dist.destroy_process_group()


def test_partition():
    assert partition(1024, 4, 0) == (0, 256) and partition(1024, 4, 3) == (768, 256)
    with pytest.raises(ValueError):
        partition(1000, 3, 0)


def test_two_rank_sharded_stepping_matches_single_process(tmp_path):
    cfg, pm, vel = inputs.make_config(1, n_override=N)
    rng = np.random.Generator(np.random.PCG64(7))
    vel = vel.copy()
    vel[:, :3] = 0.05 * rng.standard_normal((N, 3)).astype(np.float32)
    mids, _ = oracle.midstep_schedule(cfg.cosmo, cfg.a_start, cfg.tau, STEPS)
    coeffs = []
    for a, H in mids:          # eqs. (3)-(5): d1, cv, ck, d2
        coeffs.append((0.5 * cfg.tau, (1 - H * cfg.tau) / (1 + H * cfg.tau),
                       cfg.tau / (a ** 3 * (1 + H * cfg.tau)), 0.5 * cfg.tau))

    mp.spawn(_worker, args=(WORLD, _free_port(), pm, vel, float(cfg.eps2), cfg.G, coeffs, str(tmp_path)),
             nprocs=WORLD, join=True)

    ref = oracle.State(pm, vel, cfg.eps2, cfg.G)
    for c in coeffs:
        ref.step_coeffs(*c)
    pos0 = np.load(tmp_path / "pos0.npy")
    pos1 = np.load(tmp_path / "pos1.npy")
    assert np.array_equal(pos0, pos1)                      # every rank ends with the same full position array
    assert np.abs(pos0[:, :3] - ref.x).max() <= 1e-14      # same arithmetic, per-target sums in the same order
    v = np.concatenate([np.load(tmp_path / "vel0.npy"), np.load(tmp_path / "vel1.npy")])
    assert np.abs(v - ref.v).max() <= 1e-13
    assert np.array_equal(pos0[:, 3], pm[:, 3].astype(np.float64))   # masses untouched by the exchange
