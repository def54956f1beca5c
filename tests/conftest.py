"""pytest configuration: registers the `gpu` marker and puts the repo root on sys.path.

`-m "not gpu"` tests run on a CPU-only box (oracle pins, host logic, C-ABI symbol
check); `-m gpu` tests are the CUDA-vs-oracle parity tests and need one B200.
"""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def cfg0_event():
    from comet_synth import make_config
    return make_config(0)[0]


@pytest.fixture(scope="session")
def cfg1_event():
    from comet_synth import make_config
    return make_config(1)[0]
