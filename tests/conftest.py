import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

# keep the oracle's OpenMP pool and numpy from oversubscribing each other
os.environ.setdefault("OMP_NUM_THREADS", str(os.cpu_count() or 1))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "multigpu: needs two CUDA devices and NCCL (skipped, with that reason, on one)")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build_all()
    return oracle
