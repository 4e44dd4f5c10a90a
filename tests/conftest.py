import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")
    config.addinivalue_line("markers", "slow: long-running full-size check")


@pytest.fixture(scope="session")
def oracle():
    from oracle import rqa_oracle
    rqa_oracle.build()
    return rqa_oracle


@pytest.fixture(scope="session")
def rqa():
    """The CUDA path (C-ABI library through its thin Python binding).  GPU tests only."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2208_09136_b200 as pkg
    pkg.load_library()          # fails loudly if librqa.so is missing
    return pkg
