import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")
    # a leftover BEMCUB_LIB would make every parity result describe some other binary than csrc/ at HEAD
    from paper_1606_03743_b200 import build
    if build.override_refused():
        raise pytest.UsageError("BEMCUB_LIB is set (%s): the tests check the library built from csrc/; unset it, or set "
                                "BEMCUB_LIB_ALLOW=1 to test that binary on purpose" % os.environ["BEMCUB_LIB"])


def read_golden(name):
    """Rows of a whitespace-separated golden text file, '#' comments skipped."""
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                rows.append(line.split())
    return rows


@pytest.fixture(scope="session")
def golden():
    return read_golden
