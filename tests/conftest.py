"""pytest configuration: registers the `gpu` marker and puts the repo root on sys.path.

`-m "not gpu"` : oracle pins, host-side generator logic, C-ABI symbol checks (CPU only).
`-m gpu`       : parity of the CUDA path (through the C-ABI) against the oracle, on a B200.
"""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
TESTS = os.path.dirname(os.path.abspath(__file__))
if TESTS not in sys.path:
    sys.path.insert(0, TESTS)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


_ORACLE_CACHE = {}


@pytest.fixture(scope="session")
def oracle_process():
    """Factory returning cached oracle Process objects (colour construction is slow for big ones)."""
    from oracle import oracle as O

    def get(name, tier1=False):
        key = (name, tier1)
        if key not in _ORACLE_CACHE:
            _ORACLE_CACHE[key] = O.Process(name, 0.118, keep_diagram_colour=tier1)
        return _ORACLE_CACHE[key]

    return get
