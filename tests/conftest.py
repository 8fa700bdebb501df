import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session", autouse=True)
def _build_oracle():
    from oracle import psc_oracle

    psc_oracle.build()


@pytest.fixture(autouse=True)
def _dense_set_guards():
    """include/psc.h: the dense (primary) column set needs only n entries.  The harness puts
    sentinel entries behind them; after every test that built a Simulation they must be intact."""
    yield
    mod = sys.modules.get("paper_1310_7866_b200.harness")
    if mod is None:
        return
    for sim in list(mod.Simulation.live):
        assert sim.guards_intact(), "the library wrote behind the n entries of a dense column"
