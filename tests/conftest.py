import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


class _Observed:
    """Worst observed parity errors of a GPU run, beside the tolerance they were tested against.  Written to
    gpurun_out/parity_observed.txt at the end of the session (the only folder that comes back from the GPU box); the
    copy under profiles/ is what DESIGN "Tolerances" cites."""

    def __init__(self):
        self.rows = {}

    def __call__(self, name, value, tol):
        old = self.rows.get(name)
        if old is None or value > old[0]:
            self.rows[name] = (float(value), float(tol))

    def write(self):
        if not self.rows:
            return
        d = os.path.join(ROOT, "gpurun_out")
        os.makedirs(d, exist_ok=True)
        with open(os.path.join(d, "parity_observed.txt"), "w") as f:
            f.write("%-64s %12s %12s\n" % ("check", "worst", "tolerance"))
            for k in sorted(self.rows):
                f.write("%-64s %12.3e %12.3e\n" % (k, *self.rows[k]))


_OBSERVED = _Observed()


@pytest.fixture(scope="session")
def observed():
    return _OBSERVED


def pytest_sessionfinish(session, exitstatus):
    _OBSERVED.write()
