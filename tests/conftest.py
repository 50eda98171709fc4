import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def mlp_w():
    import gen
    return gen.mlp_weights(0)


@pytest.fixture(scope="session")
def orc_mlp(mlp_w):
    from oracle import ds_oracle as O
    return O.Mlp(mlp_w)
