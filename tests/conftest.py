import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a real B200 (sm_100a); run with -m gpu")


@pytest.fixture(scope="session")
def c2_W_bits():
    """The 151936 x 1536 bf16 LM-head matrix of config C2 (shared: ~6 s to draw)."""
    from paper_2606_31580_b200 import workloads as wl
    return wl.make_W(151936, 1536, 0.02, wl.SEED_BASE + 2 + wl.W_SEED_OFFSET)


@pytest.fixture(scope="session")
def tau_defaults():
    import oracle
    return oracle.TauParams()  # PAPER.md:195, paper units (L_target = 10)


@pytest.fixture(scope="session")
def tau_norm():
    import oracle
    from paper_2606_31580_b200 import workloads as wl
    return oracle.TauParams(**wl.TAU_DEFAULTS_NORMALISED)
