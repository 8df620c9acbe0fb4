import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def orc():
    from oracle import orc as _orc
    _orc.build()
    return _orc


def pytest_terminal_summary(terminalreporter):
    """Margins of the parity runs (worst Q14 against the bar), so that a `-q` log shows more than dots."""
    from tests import parity
    if parity.MARGINS:
        terminalreporter.write_sep("-", "parity margins (CUDA path vs oracle)")
        for line in parity.MARGINS:
            terminalreporter.write_line(line)
