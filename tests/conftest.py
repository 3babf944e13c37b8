import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def tables():
    import inputs
    return inputs.make_physics_tables()


@pytest.fixture(scope="session")
def oracle_c1(tables):
    """Oracle context with the 3-bin air / exact-water / Ti table (config C1 materials)."""
    import inputs
    from oracle import Oracle
    return Oracle(tables, inputs.make_materials_c1())
