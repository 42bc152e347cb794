import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: full-length parity run, opt-in with LPC_FULL=1")


@pytest.fixture(scope="session")
def oracle_mod():
    """The CPU oracle front end (oracle/lpc_oracle.py), loaded by path."""
    import importlib.util

    spec = importlib.util.spec_from_file_location("lpc_oracle", os.path.join(ROOT, "oracle", "lpc_oracle.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod
