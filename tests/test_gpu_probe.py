"""Device microbenchmarks of libcolatus_probe (include/colatus_probe.h) -- the numbers behind DESIGN.md 6.1-6.2.
They are hardware measurements, not parity tests: the bounds below are deliberately wide (a sub-cycle wobble must
never stop `pytest -x`); the measured values go to gpurun_out/parity_errors.jsonl for the record."""
import pytest

pytestmark = pytest.mark.gpu

from paper_1208_3444_b200 import probe as P  # noqa: E402
from conftest import record_parity  # noqa: E402


def test_calibrated_fp32_peak_is_near_the_derived_one():
    """148 SMs x 128 lanes x 2 flop x clock.  The register-only loops must land within
    a few percent of it at the clock the device actually runs (never above the max-clock figure)."""
    for packed in (0, 1):
        tflops, ms = P.fp32_peak(packed)
        assert ms > 0
        assert 0.70 * 74.45 <= tflops <= 1.02 * 74.45, (packed, tflops)
    assert P.lib().colatus_probe_fp32_peak(0, 0, None, None) == -1


def test_pipe_probe_issue_rules():
    """DESIGN.md 6.2, reproduced from committed code: packed FP32 ops saturate the FMA pipe at 24 SMSP cycles per
    group of 12; a broadcast LDS.128 and a MUFU are (mostly) hidden behind them, an integer add is not."""
    c = [P.pipe(m) for m in range(8)]
    record_parity("pipe probe (SMSP cycles per 12 packed ops)", ffma2=c[0], plus_2_mufu=c[1], plus_2_iadd=c[2],
                  accumulate_triples=c[3], plus_lds128=c[4], scalar_plus_2_mufu=c[5], accumulates_no_reuse=c[6],
                  plus_6_dfma=c[7])
    assert 22.0 <= c[0] <= 28.0, c
    assert c[1] <= c[0] + 5.0, c                    # MUFU: mostly hidden
    assert c[2] >= c[0] + 0.3, c                    # two integer adds: not hidden
    assert c[4] <= c[0] + 3.0, c                    # one broadcast LDS.128 per group: hidden
    assert c[5] >= c[0] - 1.0, c                    # scalar FFMA + MUFU is no faster than the packed form
    assert all(20.0 <= v <= 120.0 for v in c), c
