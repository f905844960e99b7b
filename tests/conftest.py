import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


# Build steps run before any test module is imported (the binding refuses to import without its library; the built
# .so is git-ignored): nvcc -> libgsm_b200.so, gcc -> the oracle's C helper.  Both are no-ops when up to date.
from paper_1501_01752_b200.build import build_cuda, build_oracle  # noqa: E402

build_cuda()
build_oracle()


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200)")


@pytest.fixture(scope="session", autouse=True)
def _oracle_helper():
    """The oracle's plain-C Toeplitz loop is compiled on demand (gcc); building the checker is not using it."""
    from paper_1501_01752_b200.build import build_oracle
    build_oracle()


def load_oracle_golden():
    """tests/golden/oracle_neff.txt: values written by tests/golden/make_oracle_goldens.py from the oracle alone."""
    return load_golden("oracle_neff.txt")


def load_golden(name="paper_values.txt"):
    vals = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split()
                vals[k] = float(v)
    return vals
