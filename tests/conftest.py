import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def cfg0():
    from workloads import CONFIGS
    # the pins written on this fixture are for the leaf-level reading of the hard list (T13);
    # the particle-level cut (the configs' default, R30) has its own pins in test_oracle_cut.py
    return CONFIGS[0].with_(hard_cut=0)


@pytest.fixture(scope="session")
def ic0(cfg0):
    from workloads import make_ic
    return make_ic(cfg0.kind, cfg0.n, cfg0.seed)


@pytest.fixture(scope="session")
def tree0(cfg0, ic0):
    from oracle import oracle as O
    return O.Tree(ic0[0], O.params_from(cfg0))
