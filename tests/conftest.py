import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


def pytest_sessionfinish(session, exitstatus):
    """Reading C19: the parity tests list every use of the A-floor; keep the list where gpurun brings it back."""
    mod = sys.modules.get("test_gpu_parity")
    if mod is not None and getattr(mod, "NFLOOR", None):
        import json
        out = os.path.join(ROOT, "gpurun_out")
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_floor.json"), "w") as f:
            json.dump(mod.NFLOOR, f, indent=1)
