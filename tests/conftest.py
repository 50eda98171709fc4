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


# ---- parity counts (BASELINE north_star: edge-list candidates are "listed and counted and must be < 0.01 %") ----------------
_PARITY_COUNTS = {}


@pytest.fixture(scope="session")
def parity_counts():
    """record(name, tracks=..., vertices=...) -> the counts end up in gpurun_out/parity_counts.json (or $DS_PARITY_COUNTS)."""
    def record(name, **kw):
        _PARITY_COUNTS[name] = kw
    return record


def pytest_sessionfinish(session, exitstatus):
    if not _PARITY_COUNTS:
        return
    import json
    path = os.environ.get("DS_PARITY_COUNTS", os.path.join(ROOT, "gpurun_out", "parity_counts.json"))
    try:
        os.makedirs(os.path.dirname(path), exist_ok=True)
        with open(path, "w") as f:
            json.dump(_PARITY_COUNTS, f, indent=1, sort_keys=True)
    except OSError:
        pass
