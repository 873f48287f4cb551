import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import pvref
    pvref.build()
    return pvref


@pytest.fixture(scope="session")
def cfg0():
    from synth import events
    return events.generate(events.config(0), with_truth=True)


@pytest.fixture(scope="session")
def cfg0_oracle(oracle, cfg0):
    return oracle.find(cfg0, oracle.default_params(), debug=True, n_hist_events=1000, trace=True)
