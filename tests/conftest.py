import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def load_golden(name="paper_values.txt"):
    """Parse tests/golden/<name>: 'key = value  # citation' lines -> dict of strings."""
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line or "=" not in line:
                continue
            k, v = line.split("=", 1)
            out[k.strip()] = v.strip()
    return out


@pytest.fixture(scope="session")
def golden():
    return load_golden()


# Observed parity errors: tests call record_parity(...); the numbers are printed in the terminal summary (also with -q and
# for passing tests), so the driver's log records what was actually measured, not only that it was under the gate.
PARITY_LOG = []


def record_parity(name, observed, gate):
    PARITY_LOG.append((name, float(observed), float(gate)))


@pytest.fixture(scope="session")
def parity_log():
    return record_parity


def pytest_terminal_summary(terminalreporter):
    if not PARITY_LOG:
        return
    terminalreporter.write_line("observed parity (name: observed <= gate)")
    for name, obs, gate in PARITY_LOG:
        terminalreporter.write_line(f"  {name}: {obs:.3e} <= {gate:.1e}")
