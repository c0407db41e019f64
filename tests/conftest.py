import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


@pytest.fixture(scope="session")
def mech_h2co():
    from paper_1607_03884_b200 import synth
    return synth.make_mechanism("h2co", synth.MECH_SEED)


@pytest.fixture(scope="session")
def mech_gri():
    from paper_1607_03884_b200 import synth
    return synth.make_mechanism("gri", synth.MECH_SEED)
