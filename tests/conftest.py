import os
import sys

import pytest

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def sys1():
    from workloads import make_system
    return make_system(1)


@pytest.fixture(scope="session")
def oracle1(sys1):
    from oracle.risp_oracle import Oracle
    o = Oracle(sys1)
    o.build()
    return o


@pytest.fixture(scope="session")
def sys_small_rsh():
    """12-atom cluster from the cfg-3 recipe (RSH operator, 40 eV window): small enough for an explicit A."""
    from workloads import make_system
    return make_system(3, counts=(6, 4, 1, 1))


@pytest.fixture(scope="session")
def oracle_small_rsh(sys_small_rsh):
    from oracle.risp_oracle import Oracle
    o = Oracle(sys_small_rsh)
    o.build()
    return o
