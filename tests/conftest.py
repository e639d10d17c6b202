import os
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parents[1]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def orc():
    """The CPU oracle (test infrastructure)."""
    from oracle import rbq_oracle
    rbq_oracle.build()
    return rbq_oracle


@pytest.fixture(scope="session")
def rot128(orc):
    """Dense QR rotation of the workload recipe (fp32 and fp64 copies)."""
    from paper_2606_31519_b200 import synth
    return orc.rotation_from_gaussian(synth.rotation_gaussian(128))
