import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def cfg0():
    import gen
    return gen.config0()


@pytest.fixture(scope="session")
def cfg1_small():
    """configs[1] recipe (same scene, tree depth 8, 4 levels, F=8 fp16, MLP 38->3x64->3) at a 192x160 frame."""
    import gen
    return gen.scene_workload(1, width=192, height=160)
