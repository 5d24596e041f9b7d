import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def rng_seed():
    return 20230310


# ---- measured worst cases, printed whether or not the run captures stdout ------------------------------------------------
# GPU parity tests hand their measured errors to the ``report`` fixture; the lines are echoed (visible with -s) and
# printed once more in the terminal summary, so that the numbers DESIGN.md section 6 quotes can be read from a plain
# ``pytest -q -m gpu`` log (the driver's GPUTEST record keeps the tail of that log).
_REPORT = []


@pytest.fixture
def report():
    def add(line: str):
        _REPORT.append(line)
        print(line)
    return add


def pytest_terminal_summary(terminalreporter):
    if _REPORT:
        terminalreporter.write_sep("-", "parity report: measured errors (tolerances: forward 1e-4 |F(0)|, gradient 1e-3 rel L2, image 1e-4 max)")
        for line in _REPORT:
            terminalreporter.write_line(line)
