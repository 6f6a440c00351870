"""pytest configuration: registers the `gpu` marker (tests that need a B200) and a few shared fixtures."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def geom():
    from paper_1908_01949_b200 import synth
    return synth.make_geometry()


@pytest.fixture(scope="session")
def uniform_field():
    from paper_1908_01949_b200 import synth
    return synth.make_uniform_field()


@pytest.fixture(scope="session")
def table_field():
    from paper_1908_01949_b200 import synth
    return synth.make_table_field()
