import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200, sm_100a)")


@pytest.fixture(scope="session")
def c1_inputs():
    from paper_2607_07724_b200 import synth
    return synth.make_inputs(synth.CONFIGS["C1"])


@pytest.fixture(scope="session")
def c1_meta(c1_inputs):
    import oracle
    return oracle.pool(c1_inputs.K, c1_inputs.cfg.block)
