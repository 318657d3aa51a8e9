import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def swave_table():
    from oracle import channels, perm

    ch, pairs = channels.spinless_swave_table(1.0)
    return perm.PairTable(ch, pairs)


@pytest.fixture(scope="session")
def nd_half_plus_j1():
    """J^pi = 1/2+, pair j <= 1: 10 channels, l <= 2 -- small multichannel table."""
    from oracle import channels, perm

    ch = channels.enumerate_channels(1, +1, 1)
    return perm.PairTable(ch, channels.g_table(ch, 1, 1))


@pytest.fixture(scope="session")
def wpcd():
    """The product binding, with libwpcd.so (re)built in-tree if sources are newer."""
    from paper_1404_5253_b200 import build as _build

    _build.build()
    import paper_1404_5253_b200 as mod

    mod.load()
    return mod
