"""Target-sharded multi-GPU stepping.

Eq. (1) shards by TARGETS: every rank holds all n sources, owns a contiguous slice of the
particles, evaluates forces / drifts / kicks for its slice only (libcolatus target range) and the
ranks exchange updated positions with one all-gather after each drift -- the path's only real
exchange step.  One process per GPU; `torch.distributed` (NCCL over NVLink on GPUs, gloo in the
CPU tests) is the plumbing.

`ShardedStepper` holds only the host-side sequencing.  The per-slice work is done by an `ops`
object: `LibcolatusOps` (the product: calls the C ABI) or, in tests/, a stand-in that lets the
sequencing be checked on CPU without a GPU.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def partition(n: int, world: int, rank: int):
    """Contiguous equal slices; n must be a multiple of world (the all-gather is in place)."""
    if n % world != 0:
        raise ValueError(f"n={n} is not a multiple of world size {world}")
    c = n // world
    return rank * c, c


class LibcolatusOps:
    """Per-slice work through the C ABI on the resident state (pos, vel device tensors)."""

    def __init__(self, pos, vel, acc_slice, n, eps2, begin, count):
        from . import binding as B
        self.B = B
        B.colatus_upload(pos, vel, acc_slice, n, eps2)
        B.colatus_set_target_range(begin, count)

    def drift(self, d):
        self.B.colatus_drift(d)

    def force_kick_drift(self, cv, ck, d2):
        self.B.colatus_force_kick_drift(cv, ck, d2)


class ShardedStepper:
    def __init__(self, pos: torch.Tensor, n: int, ops, group=None):
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.group = group
        self.pos = pos                       # [n,4] full body array, identical on all ranks at step ends
        self.n = n
        self.begin, self.count = partition(n, self.world, self.rank)
        self.ops = ops

    def _allgather_positions(self):
        if self.world == 1:
            return
        mine = self.pos[self.begin:self.begin + self.count]
        if self.pos.is_cuda:
            dist.all_gather_into_tensor(self.pos, mine, group=self.group)      # in place (NCCL)
        else:
            parts = [torch.empty_like(mine) for _ in range(self.world)]
            dist.all_gather(parts, mine.clone(), group=self.group)
            for r, p in enumerate(parts):
                self.pos[r * self.count:(r + 1) * self.count].copy_(p)

    def step_coeffs(self, d1, cv, ck, d2):
        """x += d1 v | all-gather x | F, v = cv v + ck F, x += d2 v | all-gather x."""
        self.ops.drift(d1)
        self._allgather_positions()
        self.ops.force_kick_drift(cv, ck, d2)
        self._allgather_positions()

    def step(self, tau, a, H):
        """Eqs. (3)-(5), with the coefficients libcolatus forms."""
        from . import binding as B
        self.step_coeffs(*B.colatus_step_coefficients(tau, a, H))
