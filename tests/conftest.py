import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def water_tables():
    from paper_1101_1245_b200.inputs import materials as M
    from paper_1101_1245_b200.inputs.tables import build_tables
    return build_tables([M.WATER])


@pytest.fixture(scope="session")
def slab_tables():
    from paper_1101_1245_b200.inputs import materials as M
    from paper_1101_1245_b200.inputs.tables import build_tables
    return build_tables([M.WATER, M.BONE, M.LUNG])
