import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def orc():
    import oracle
    oracle.build()
    return oracle


def pytest_sessionfinish(session, exitstatus):
    """GPU parity runs: dump what the TMSE slack was worth (tests/test_gpu_parity.py PARITY_LOG) to $GAME_PARITY_LOG."""
    path = os.environ.get("GAME_PARITY_LOG")
    mod = sys.modules.get("test_gpu_parity") or sys.modules.get("tests.test_gpu_parity")
    if not path or mod is None or not getattr(mod, "PARITY_LOG", None):
        return
    import json
    with open(path, "w") as f:
        for rec in mod.PARITY_LOG:
            f.write(json.dumps(rec) + "\n")
