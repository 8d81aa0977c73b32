import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


def read_golden(name):
    """Parse a tests/golden/*.txt fixture: '#' comments, whitespace-separated columns."""
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


def pytest_terminal_summary(terminalreporter):
    """DESIGN.md R21: how many carriers used the close-encounter excuse, over all trajectory checks of the session."""
    try:
        from util import EXCUSED
    except Exception:
        return
    if not EXCUSED:
        return
    log = os.environ.get("GCORECCD_EXCUSE_LOG")
    if log:
        with open(log, "w") as f:
            for e in EXCUSED:
                f.write("%d %d %s %s ext=%d knock=%d\n" % (e[2], e[1], e[0], e[3], e[4] if len(e) > 4 else 0, e[5] if len(e) > 5 else 0))
    tot = sum(e[1] for e in EXCUSED)
    exc = sum(e[2] for e in EXCUSED)
    terminalreporter.write_line("R21 excuse clause: %d trajectory checks, %d carriers compared, %d excused (%.4f %%); "
                                "largest single check: %d; R21b extended radius: %d, knock-on: %d"
                                % (len(EXCUSED), tot, exc, 100.0 * exc / max(tot, 1), max(e[2] for e in EXCUSED),
                                   sum(e[4] for e in EXCUSED if len(e) > 4), sum(e[5] for e in EXCUSED if len(e) > 5)))
