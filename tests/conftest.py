import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for _p in (ROOT, os.path.join(ROOT, "tests")):
    if _p not in sys.path:
        sys.path.insert(0, _p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def orc():
    from oracle import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session", autouse=True)
def _gradient_bar_log():
    """After a GPU session: what share of each gradient group lay outside the literal 1e-3 / 1e-5 tolerance and how large a
    rounding allowance c those elements needed (tests/gpu_util.compare_grads) -> gpurun_out/gradient_bar.json (scratch; the
    committed summary is profiles/r3_gradient_bar.md)."""
    yield
    try:
        import json
        import gpu_util
        if gpu_util.BAR_LOG:
            os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
            with open(os.path.join(ROOT, "gpurun_out", "gradient_bar.json"), "w") as f:
                json.dump(gpu_util.BAR_LOG, f, indent=0)
    except Exception:      # never fail a test session over the log
        pass
