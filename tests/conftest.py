import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def load_golden():
    """Parse tests/golden/shift_pins.txt (values cited from SURVEY.md §8(c))."""
    pins, dm30, nsamp_in = {}, {}, {}
    with open(os.path.join(ROOT, "tests", "golden", "shift_pins.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            tok = line.split()
            if tok[0] == "c1_dm30":
                dm30 = {int(k): int(v) for k, v in (p.split(":") for p in tok[1:])}
            elif tok[0] == "nsamp_in":
                nsamp_in[tok[1]] = int(tok[2])
            else:
                pins[tok[0]] = tuple(int(x) for x in tok[1:])
    return pins, dm30, nsamp_in


@pytest.fixture(scope="session")
def golden():
    return load_golden()
