import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


_structs = {}


@pytest.fixture(scope="session")
def oracle_structures():
    """Session cache of oracle fold libraries (6x6 and 3x3x3 take tens of seconds to enumerate)."""
    from oracle import gp_oracle

    def get(nx, ny, nz=1):
        key = (nx, ny, nz)
        if key not in _structs:
            _structs[key] = gp_oracle.Structures(nx, ny, nz)
        return _structs[key]
    return get
