import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

GOLDEN = Path(__file__).resolve().parent / "golden"


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: full-size parity run (minutes; opt-in through CS_FULL_PARITY=1)")


@pytest.fixture(scope="session")
def golden():
    import json
    with open(GOLDEN / "pins.json") as f:
        return json.load(f)
