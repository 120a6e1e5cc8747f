"""Convenience driver over `binding`: owns the torch device buffers and the workspace and walks
the Appendix-A sequence of the paper (allocate, copy H2D, loop steps, copy back).

No arithmetic of the method happens here: forces, drifts, kicks, tracer records and reductions
all run in libcolatus kernels; the scale factor schedule comes from the library's host helpers
(eq. (2)).  Requires a CUDA device -- there is no CPU path.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as B


class Session:
    """One libcolatus context (the library has a single process-wide context)."""

    def __init__(self, G: float, n_max: int, device: int = 0):
        if not torch.cuda.is_available():
            raise B.ColatusError(B.CUDA_ERROR, "no CUDA device: libcolatus has no CPU fallback")
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self.n_max = int(n_max)
        self.workspace = torch.empty(B.colatus_workspace_bytes(n_max), dtype=torch.uint8, device=self.device)
        B.colatus_init(G, device, self.workspace)
        self.G = float(G)
        self._open = True
        self.pos = self.vel = self.acc = None
        self.ring = self.trace_idx = None

    def close(self):
        if self._open:
            torch.cuda.synchronize()
            B.colatus_shutdown()
            self._open = False

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # ---- eq. (1) ------------------------------------------------------------------------------
    def to_device(self, arr: np.ndarray) -> torch.Tensor:
        return torch.from_numpy(np.ascontiguousarray(arr, dtype=np.float32)).to(self.device)

    def forces(self, pos_mass, eps2, potential=False, target_range=None) -> torch.Tensor:
        """pos_mass: float32 [n,4] numpy array or CUDA tensor.  Returns a CUDA tensor [k,4]."""
        pm = pos_mass if isinstance(pos_mass, torch.Tensor) else self.to_device(pos_mass)
        n = pm.shape[0]
        if target_range is None:
            out = torch.empty((n, 4), dtype=torch.float32, device=self.device)
            (B.colatus_forces_potential if potential else B.colatus_forces)(pm, n, eps2, out)
        else:
            b, c = target_range
            out = torch.empty((c, 4), dtype=torch.float32, device=self.device)
            B.colatus_forces_range(pm, n, b, c, eps2, out)
        return out

    # ---- eqs. (3)-(5) --------------------------------------------------------------------------
    def upload(self, pos_mass: np.ndarray, vel: np.ndarray, eps2):
        self.pos = self.to_device(pos_mass)
        self.vel = self.to_device(vel)
        self.acc = torch.zeros_like(self.pos)
        self.n = self.pos.shape[0]
        B.colatus_upload(self.pos, self.vel, self.acc, self.n, eps2)

    def trace(self, idx: np.ndarray, capacity_steps: int):
        self.trace_idx = torch.from_numpy(np.ascontiguousarray(idx, dtype=np.int32)).to(self.device)
        k = int(self.trace_idx.numel())
        self.ring = torch.zeros((capacity_steps, k, 4), dtype=torch.float32, device=self.device)
        B.colatus_trace(self.trace_idx, k, self.ring, capacity_steps)
        self.trace_k = k

    def trace_read(self, first_step: int, n_steps: int) -> np.ndarray:
        out = np.empty((n_steps, self.trace_k, 4), dtype=np.float32)
        B.colatus_trace_read(out, first_step, n_steps)
        return out

    def run(self, cosmo, a_start: float, tau: float, steps: int):
        """`steps` steps of eqs. (3)-(5) with a, H at mid-step (reading G3) from the library's own
        Friedmann helpers; cosmo None = static background (a=1, H=0).  Returns a at the end."""
        a = float(a_start)
        for _ in range(steps):
            if cosmo is None:
                B.colatus_step(tau, 1.0, 0.0)
            else:
                a_mid = B.colatus_a_advance(cosmo, a, 0.5 * tau)
                B.colatus_step(tau, a_mid, B.colatus_hubble(cosmo, a_mid))
                a = B.colatus_a_advance(cosmo, a_mid, 0.5 * tau)
        return a

    def run_native(self, cosmo, a_start: float, tau: float, steps: int, use_graph: bool = True):
        """The same steps as `run`, in one colatus_run call (native loop, CUDA-graph replay)."""
        return B.colatus_run(cosmo, a_start, tau, steps, use_graph)

    def download(self):
        pos = np.empty((self.n, 4), dtype=np.float32)
        vel = np.empty((self.n, 4), dtype=np.float32)
        B.colatus_download(pos, vel)
        return pos, vel

    def diagnostics(self, a=1.0, with_potential=False):
        return np.array(B.colatus_diagnostics(a, with_potential))

    # ---- NEXT rows f4, f3: snapshot image and tracer spectrum ------------------------------------------
    def splat(self, axis, window, width, height, pos_mass=None) -> np.ndarray:
        """Particle-count image uint32 [height, width] of `pos_mass` (numpy / CUDA tensor) or, if None,
        of the resident positions."""
        img = torch.empty((height, width), dtype=torch.int32, device=self.device)
        pm = None
        if pos_mass is not None:
            pm = pos_mass if isinstance(pos_mass, torch.Tensor) else self.to_device(pos_mass)
        B.colatus_splat(pm, 0 if pm is None else pm.shape[0], axis, window, width, height, img)
        return img.cpu().numpy().view(np.uint32)

    def trace_spectrum(self, first_step: int, n_steps: int) -> np.ndarray:
        out = torch.empty((self.trace_k, n_steps // 2 + 1), dtype=torch.float64, device=self.device)
        B.colatus_trace_spectrum(first_step, n_steps, out)
        return out.cpu().numpy()
