import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def golden_dir():
    return ROOT / "tests" / "golden"


def pytest_sessionfinish(session, exitstatus):
    """GPU parity runs: keep the achieved errors of every compared iteration and the "reported separately" list
    (tests/parity.py) in gpurun_out/parity_stats.txt -- all test modules of the session."""
    Pz = sys.modules.get("parity")
    if Pz is None or not getattr(Pz, "STATS", None):
        return
    out = ROOT / "gpurun_out"
    if out.is_dir():
        (out / "parity_stats.txt").write_text("\n".join(Pz.STATS + ["", "reported separately:"] + Pz.REPORT) + "\n")
    if Pz.REPORT:
        print("\n[parity] reported separately:\n  " + "\n  ".join(Pz.REPORT))
