"""Multi-GPU stepping: bodies are owned in contiguous slices; eq. (1) is
divided either by TARGETS (every rank evaluates the forces on its own slice with the one-directional kernel) or, for
problems large enough for the symmetric kernel, by BLOCK PAIRS (every rank evaluates its share of the unordered pairs
once and one all-reduce of the float4[n] partial forces delivers action and reaction to their owners).

Eq. (1) shards by TARGETS: every rank holds all n sources, owns a contiguous slice of the
particles, evaluates forces / drifts / kicks for its slice only (libcolatus target range) and the
ranks exchange updated positions with ONE all-gather per step, after the first half drift -- the
path's only real exchange step (it replaces the paper's per-step device-to-host copy of everything,
PAPER.md:116).  After the kick-drift a rank's copy of the OTHER slices is stale; nothing needs them
until the next step's all-gather, so the stepper only marks the positions dirty and gathers lazily
before a read of full positions (`sync_positions`: download, potential energy).  Diagnostics are one
all-reduce of 16 doubles; a tracer's velocity row is recorded by the rank that owns the particle and
the rows are assembled on read.  One process per GPU; `torch.distributed` (NCCL over NVLink on GPUs,
gloo in the CPU tests) is the plumbing.

Symmetric mode (`symmetric=True`, the default from SYMMETRIC_MIN_N bodies on when the ops object supports it): the
force step of a rank is `ops.forces_symmetric_part(rank, world, acc_full)` -- the block pairs whose target block lies
in the rank's share, circulant pairing so every share is the same work, every pair evaluated once -- followed by ONE
all-reduce (sum) of acc_full (16 n bytes: 16 MiB at 2^20, microseconds over NVLink against 314 ms / world of force
work), `ops.add_external(acc_full[slice])` (the eq. (10) source and the background term, which a share cannot carry:
once, on the sum) and `ops.kick_drift(acc_full[slice], ...)`.  Per step: one all-gather of positions and one all-reduce of forces.

`ShardedStepper` holds only the host-side sequencing.  The per-slice work is done by an `ops`
object: `LibcolatusOps` (the product: calls the C ABI) or, in tests/, a stand-in that lets the
sequencing be checked on CPU without a GPU.  An `ops` object provides
    drift(d); force_kick_drift(cv, ck, d2); diagnostics(a, with_potential) -> 16 doubles over the slice;
    trace_rows(first_step, n_steps) -> float32 [n_steps, k, 4] of this rank's ring (optional);
    forces_symmetric_part(part, parts, acc_full); add_external(acc_slice); kick_drift(acc_slice, cv, ck, d2)
    (optional: symmetric mode).
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist


SYMMETRIC_MIN_N = 20480          # as libcolatus: below, the one-directional kernel on target slices is faster


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
        self.trace_k = 0
        self.pos, self.n, self.eps2 = pos, n, eps2
        B.colatus_upload(pos, vel, acc_slice, n, eps2)
        B.colatus_set_target_range(begin, count)

    def drift(self, d):
        self.B.colatus_drift(d)

    def force_kick_drift(self, cv, ck, d2):
        self.B.colatus_force_kick_drift(cv, ck, d2)

    def forces_symmetric_part(self, part, parts, acc_full):
        """acc_full: float32 device tensor [n, 4]; receives this share's partial forces on ALL bodies."""
        self.B.colatus_forces_symmetric_part(self.pos, self.n, self.eps2, part, parts, acc_full)

    def kick_drift(self, acc_slice, cv, ck, d2):
        self.B.colatus_kick_drift(acc_slice, cv, ck, d2)

    def add_external(self, acc_slice):
        """eq. (10) source / background term, once, on the summed forces of the own slice (no launch when both are off)."""
        self.B.colatus_add_external(acc_slice)

    def diagnostics(self, a, with_potential=False):
        return self.B.colatus_diagnostics(a, with_potential)

    def trace(self, idx_dev, ring_dev, capacity_steps):
        """idx_dev: int32 device tensor [k] (global particle indices); ring_dev: float32 device tensor
        [capacity_steps, k, 4].  Only the tracers inside this rank's slice are ever written."""
        self.trace_k = int(idx_dev.numel())
        self.B.colatus_trace(idx_dev, self.trace_k, ring_dev, capacity_steps)

    def trace_rows(self, first_step, n_steps):
        out = np.empty((n_steps, self.trace_k, 4), dtype=np.float32)
        self.B.colatus_trace_read(out, first_step, n_steps)
        return out


class ShardedStepper:
    def __init__(self, pos: torch.Tensor, n: int, ops, group=None, symmetric=None):
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.group = group
        self.pos = pos                       # [n,4] full body array; other ranks' slices may be stale (dirty)
        self.n = n
        self.begin, self.count = partition(n, self.world, self.rank)
        self.ops = ops
        self.dirty = False                   # True: the slices owned by other ranks are not current here
        self.gathers = 0                     # all-gathers issued (one per step + lazy syncs)
        if symmetric is None:
            symmetric = n >= SYMMETRIC_MIN_N and hasattr(ops, "forces_symmetric_part")
        self.symmetric = bool(symmetric)
        self.acc_full = torch.zeros_like(pos) if self.symmetric else None      # [n,4] partial / reduced forces
        self.reduces = 0                     # force all-reduces issued (symmetric mode: one per step)

    def _allgather_positions(self):
        self.dirty = False
        if self.world == 1:
            return
        self.gathers += 1
        mine = self.pos[self.begin:self.begin + self.count]
        if self.pos.is_cuda:
            dist.all_gather_into_tensor(self.pos, mine, group=self.group)      # in place (NCCL)
        else:
            parts = [torch.empty_like(mine) for _ in range(self.world)]
            dist.all_gather(parts, mine.clone(), group=self.group)
            for r, p in enumerate(parts):
                self.pos[r * self.count:(r + 1) * self.count].copy_(p)

    def sync_positions(self):
        """Make every rank's full position array current (no-op unless a step has run since the last gather)."""
        if self.dirty:
            self._allgather_positions()

    def step_coeffs(self, d1, cv, ck, d2):
        """x += d1 v (own slice) | all-gather x | F, v = cv v + ck F, x += d2 v (own slice).
        F: the own slice's forces by the one-directional kernel, or (symmetric mode) this rank's share of the
        unordered pairs on all bodies, summed over the ranks by one all-reduce."""
        self.ops.drift(d1)
        self._allgather_positions()
        if self.symmetric:
            self.ops.forces_symmetric_part(self.rank, self.world, self.acc_full)
            if self.world > 1:
                self.reduces += 1
                dist.all_reduce(self.acc_full, op=dist.ReduceOp.SUM, group=self.group)
            mine = self.acc_full[self.begin:self.begin + self.count]
            if hasattr(self.ops, "add_external"):      # shares carry no external terms: once, after the sum
                self.ops.add_external(mine)
            self.ops.kick_drift(mine, cv, ck, d2)
        else:
            self.ops.force_kick_drift(cv, ck, d2)
        self.dirty = self.world > 1

    def step(self, tau, a, H):
        """Eqs. (3)-(5), with the coefficients libcolatus forms."""
        from . import binding as B
        self.step_coeffs(*B.colatus_step_coefficients(tau, a, H))

    def diagnostics(self, a, with_potential=False):
        """colatus_diagnostics over all n bodies: every rank reduces its own slice (out[0..8], out[13..15] are
        additive over slices), then ONE all-reduce of the 16 doubles; centre of mass = sum m x / M afterwards.
        W needs every rank's sources to be current, so the positions are synchronised first."""
        if with_potential:
            self.sync_positions()
        d = np.array(self.ops.diagnostics(a, with_potential), dtype=np.float64)
        step = d[12]
        if self.world > 1:
            t = torch.from_numpy(d.copy())
            if self.pos.is_cuda:
                t = t.to(self.pos.device)
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
            d = t.cpu().numpy()
        # the one line of the method's arithmetic outside the library: colatus_diagnostics forms the centre of mass as
        # out[13..15] / out[0] per GPU; over ranks the same FP64 division has to follow the all-reduce of both sums
        d[9:12] = d[13:16] / d[0]
        d[12] = step
        return d

    def trace_read(self, idx, first_step, n_steps):
        """Rows [first_step, +n_steps) of the tracer record, float32 [n_steps, k, 4], assembled from the ranks
        that own each tracer (idx: the global particle indices given to `ops.trace`)."""
        rows = self.ops.trace_rows(first_step, n_steps)
        if self.world == 1:
            return rows
        idx = np.asarray(idx, dtype=np.int64)
        mine = (idx >= self.begin) & (idx < self.begin + self.count)
        rows = np.where(mine[None, :, None], rows, np.float32(0.0))            # exact: owners' values + zeros
        t = torch.from_numpy(np.ascontiguousarray(rows))
        if self.pos.is_cuda:
            t = t.to(self.pos.device)
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
        return t.cpu().numpy()
