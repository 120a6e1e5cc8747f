import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


def pytest_collection_modifyitems(config, items):
    # GPU tests are deselected by `-m "not gpu"`; when selected without a device they fail loudly
    # inside the binding (no CPU fallback exists), which is the intended behaviour.
    return


@pytest.fixture(scope="session", autouse=True)
def _built_in_tree():
    """Both shared libraries are git-ignored build products: (re)build them in-tree when missing or stale, so
    that a fresh checkout runs the CUDA path (nvcc cross-compiles without a GPU) instead of failing to import."""
    from paper_1208_3444_b200 import build as cuda_build
    cuda_build.build()
    import oracle
    oracle.build()


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")


def record_parity(name, **values):
    """Append measured GPU-vs-oracle errors to gpurun_out/parity_errors.jsonl (scratch; the numbers quoted in
    DESIGN.md come from it).  Never influences a test outcome."""
    import json
    try:
        d = os.path.join(ROOT, "gpurun_out")
        os.makedirs(d, exist_ok=True)
        with open(os.path.join(d, "parity_errors.jsonl"), "a") as f:
            f.write(json.dumps({"case": name, **{k: float(v) for k, v in values.items()}}) + "\n")
    except OSError:
        pass
