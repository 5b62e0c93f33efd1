import os
import sys
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")
    config.addinivalue_line("markers", "slow: CPU test that takes more than a few seconds")


@pytest.fixture(scope="session")
def config1():
    import dvx_scenes
    return dvx_scenes.make_config(1)


@pytest.fixture(scope="session")
def config3():
    import dvx_scenes
    return dvx_scenes.make_config(3)


def pytest_terminal_summary(terminalreporter):
    """Parity notes (how many pixels each test compared and how many threshold-ambiguous pixels it had to use)."""
    try:
        from helpers import NOTES
    except ImportError:
        return
    if NOTES:
        terminalreporter.write_sep("-", "parity notes")
        for line in NOTES:
            terminalreporter.write_line(line)
