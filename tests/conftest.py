import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


# MPR_B200_LIB=<path> runs the suite against another build of the library, e.g. the -DMPR_CHECKED one
# (paper_1811_01604_b200.build.build_checked(): bounds assertions in the tile passes; profiles/r02d)
if os.environ.get("MPR_B200_LIB"):
    from paper_1811_01604_b200 import mpr as _mpr
    _mpr.LIB_PATH = os.path.abspath(os.environ["MPR_B200_LIB"])


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "slow: longer statistical test")


@pytest.fixture(scope="session")
def orc():
    """The CPU oracle (test infrastructure)."""
    from oracle import mpr_oracle
    mpr_oracle.lib()
    return mpr_oracle
