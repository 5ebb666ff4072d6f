import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def cfg1():
    import gen
    c = gen.make_config(1)
    m = c["model"]
    c["blob"] = gen.make_weights(m["n_species"], m["F"], m["K"], m["T"], m["rc"], seed=m["wseed"])
    return c
