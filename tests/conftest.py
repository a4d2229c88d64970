import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


@pytest.fixture(scope="session")
def geom_barrel():
    import lstgen
    return lstgen.build_geometry(True)


@pytest.fixture(scope="session")
def geom_full():
    import lstgen
    return lstgen.build_geometry(False)


@pytest.fixture(scope="session")
def map_barrel(geom_barrel):
    from oracle import lst_oracle as O
    return O.build_module_map(geom_barrel)


@pytest.fixture(scope="session")
def map_full(geom_full):
    from oracle import lst_oracle as O
    return O.build_module_map(geom_full)
