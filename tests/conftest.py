import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: full-size case, several minutes")


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")


def record_error(name: str, value: float, tol: float):
    """Append a measured parity error to gpurun_out/parity_errors.tsv (kept beside the GPU test log)."""
    out = os.path.join(ROOT, "gpurun_out")
    try:
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_errors.tsv"), "a") as f:
            f.write(f"{name}\t{value:.3e}\t{tol:.1e}\n")
    except OSError:
        pass
