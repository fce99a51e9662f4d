import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: full-size parity (minutes of oracle time)")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.lib()
    return oracle


_REPORT = {}


@pytest.fixture
def report():
    """report(name, line): a test hands over a line of a measured table (error classes, kernel times).  Tests
    only assert; nothing is written unless the run was started with FREDEC_TEST_REPORT=<directory>, the named
    command behind the tables summarised under profiles/."""
    def add(name, line):
        _REPORT.setdefault(name, []).append(line)
    return add


def pytest_sessionfinish(session, exitstatus):
    out = os.environ.get("FREDEC_TEST_REPORT")
    if not out or not _REPORT:
        return
    os.makedirs(out, exist_ok=True)
    for name, lines in _REPORT.items():
        with open(os.path.join(out, name + ".txt"), "w") as fh:
            fh.write("\n".join(lines) + "\n")
