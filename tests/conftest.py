import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import pimpc_oracle
    pimpc_oracle.build()
    return pimpc_oracle


def pytest_sessionfinish(session, exitstatus):
    """Observed parity margins of the session (worst iterate error, worst relative c error, replays per test label)
    -> gpurun_out/parity_stats.json, the numbers DESIGN.md section 3 quotes."""
    from tests import parity
    if not parity.STATS:
        return
    import json
    out = os.path.join(ROOT, "gpurun_out")
    try:
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_stats.json"), "w") as f:
            json.dump(parity.STATS, f, indent=1, sort_keys=True)
    except OSError:
        pass
