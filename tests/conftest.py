import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def tiny_arch():
    from synth_inputs import Arch
    # L=2, d=32, 4 query heads / 2 KV heads x 8, FFN 48, vocab 64, logits x8
    return Arch(2, 32, 4, 2, 8, 48, 64, 63, 0, 8.0, 1e-5, 10000.0, 0.02)
