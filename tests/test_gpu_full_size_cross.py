"""BASELINE configs 4 and 5 at their full size: every target through both force kernels (see the test's docstring).
A module of its own: it needs a library session sized for 2^22 bodies."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1208_3444_b200 import binding as B  # noqa: E402
from paper_1208_3444_b200 import inputs  # noqa: E402
from conftest import record_parity  # noqa: E402


@pytest.mark.parametrize("index", [4, 5])
def test_full_size_both_kernels_agree_on_every_target(index):
    """BASELINE configs 4 (N = 2^20, the launch configuration bench.py times: 256 blocks of 4096 bodies, 8 launches of
    17 block distances) and 5 (N = 2^22: 1024 blocks, 27 launches): the oracle can check 4096 sampled targets (test_gpu_forces.py);
    here EVERY target is compared between the symmetric and the one-directional kernel -- two independent
    decompositions of eq. (1) -- so that no block, tile, split or chunk boundary of the full-size geometry can hide
    between the samples."""
    import torch
    from paper_1208_3444_b200.harness import Session
    cfg, pm, _ = inputs.make_config(index)
    with Session(1.0, cfg.n) as s:
        d = s.to_device(pm)
        plan = B.colatus_force_plan(cfg.n)
        # 32 partial rows per launch (the row budget, profiles/r03_workspace_rows_sweep.md): 15 / 13 splits + 17 / 19 distances
        assert plan["symmetric"] == 1 and plan["blocks"] == cfg.n // 4096 and plan["partial_rows"] == 32
        assert plan["launches"] == {4: 8, 5: 27}[index], plan
        sym = s.forces(d, cfg.eps2)
        B.colatus_set_option("symmetric", 0)
        plain = s.forces(d, cfg.eps2)
        B.colatus_set_option("symmetric", 1)
        diff = (sym[:, :3].double() - plain[:, :3].double()).norm(dim=1)
        nr = plain[:, :3].double().norm(dim=1)
        med = float((diff / nr).median())
        mx = float(diff.max() / (nr ** 2).mean().sqrt())
        worst_rel = float((diff / nr).max())
        torch.cuda.synchronize()
    record_parity(f"config {index}: symmetric vs one-directional kernel, all targets", n=cfg.n, targets=cfg.n,
                  median_rel=med, max_over_rms=mx, worst_rel=worst_rel)
    assert med <= 2e-6 and mx <= 2e-5, (med, mx)
