import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def orc():
    import oracle

    oracle.build()
    return oracle


def pytest_sessionfinish(session, exitstatus):
    """PASTA_PARITY_STATS=<file>: dump what the GPU parity tests measured (per-seed trajectory errors, D22 rescues,
    evolved-snapshot force errors) as JSON, for profiles/."""
    path = os.environ.get("PASTA_PARITY_STATS")
    mod = sys.modules.get("test_gpu_parity") or sys.modules.get("tests.test_gpu_parity")
    if not path or mod is None:
        return
    import json

    with open(path, "w") as f:
        json.dump({"trajectory": mod.TRAJ, "d22_rescued": mod.RESCUED,
                   "evolved": [dict(zip(("cfg", "step", "density", "rel_l2", "worst_particle"), e)) for e in mod.EVOLVED]},
                  f, indent=1)
