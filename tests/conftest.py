import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")
    config.addinivalue_line("markers", "slow: full-size oracle comparisons (minutes of host time)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import lcf_oracle
    lcf_oracle.build()
    return lcf_oracle
