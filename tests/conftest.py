import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle_ld():
    from oracle.sc_oracle import Oracle
    return Oracle("ld")


@pytest.fixture(scope="session")
def oracle_plain():
    from oracle.sc_oracle import Oracle
    return Oracle("plain")


@pytest.fixture(scope="session")
def scmd():
    """The CUDA library binding; fails loudly if libscmd.so is missing."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1210_3559_b200 as pkg
    pkg.load_library()
    return pkg
