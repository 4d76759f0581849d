import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def wl():
    from paper_1503_01725_b200 import workloads
    return workloads


@pytest.fixture(scope="session")
def orc():
    import oracle
    oracle.lib()
    return oracle


@pytest.fixture(scope="session")
def cfg(wl):
    cache = {}

    def get(name, with_phantom=True):
        key = (name, with_phantom)
        if key not in cache:
            cache[key] = wl.make_config(name, with_phantom=with_phantom)
        return cache[key]
    return get


@pytest.fixture(scope="session")
def opsl(orc, cfg):
    cache = {}

    def get(name):
        if name not in cache:
            c = cfg(name, with_phantom=False)
            cache[name] = orc.Psl(c["psr"], c["jaws"], c["n_sectors"])
        return cache[name]
    return get
