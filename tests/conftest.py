import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def orc():
    """Long-double CPU oracle (the parity truth)."""
    from oracle.binding import Oracle
    return Oracle("ld")


@pytest.fixture(scope="session")
def orc_d():
    """fp64 instantiation of the same oracle source (the fp64 rounding floor)."""
    from oracle.binding import Oracle
    return Oracle("d")


class _ParityRecord:
    """Collects what the GPU parity tests measure -- per config, case and channel: raw rel-L2 against
    the long-double oracle, the error relative to the common scale of the three channels, the fp64
    rounding floor (the oracle's own fp64 build against its long-double build, where computed), the
    bar and pass/fail -- and writes it as JSON when the session ends (report the raw number,
    the common-scale number and the measured floor, and state pass/fail for each).
    Path: $LISA_TD_PARITY_OUT, default gpurun_out/parity_record.json."""

    def __init__(self):
        self.rows = []

    def __call__(self, config, case, quantity, raw=None, common=None, floor=None, tol=None, passed=None, note=None):
        f = lambda v: None if v is None else float(v)
        self.rows.append(dict(config=config, case=case, quantity=quantity, raw_rel_l2=f(raw), vs_common_scale=f(common),
                              fp64_floor=f(floor), bar=f(tol), passed=None if passed is None else bool(passed), note=note))

    def dump(self):
        if not self.rows:
            return
        import json
        path = os.environ.get("LISA_TD_PARITY_OUT", os.path.join(ROOT, "gpurun_out", "parity_record.json"))
        try:
            os.makedirs(os.path.dirname(path), exist_ok=True)
            with open(path, "w") as fh:
                json.dump({"north_star_bars": {"tdi_rel_l2_per_channel": 1e-11, "loglike_relative": 1e-9},
                           "truth": "oracle/lisa_oracle.c, long-double build; floor = its fp64 build against it",
                           "rows": self.rows}, fh, indent=1)
        except OSError:
            pass


_PARITY = _ParityRecord()


@pytest.fixture(scope="session")
def parity_record():
    return _PARITY


def pytest_sessionfinish(session, exitstatus):
    _PARITY.dump()
