import os
import sys

import pytest

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: takes more than a few seconds")


@pytest.fixture(scope="session")
def cfg1():
    """BASELINE.json config 1 with its 2^24 brute-force energies (about 10 s, once per session)."""
    import instances
    from oracle import brute
    inst, run = instances.config(0)
    return inst, run, brute.all_energies(inst)
