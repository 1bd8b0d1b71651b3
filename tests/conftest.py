import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def oracle():
    from oracle import sparda_oracle

    sparda_oracle.build()
    return sparda_oracle


# "count and report how many rows used the band" -- per test, in the terminal summary (-m gpu runs)
_band_by_test = {}


@pytest.hookimpl(hookwrapper=True)
def pytest_runtest_call(item):
    import parity
    n0 = len(parity.BAND_LOG)
    yield
    new = parity.BAND_LOG[n0:]
    if new:
        _band_by_test[item.nodeid] = (sum(r for r, _ in new), sum(b for _, b in new))


def pytest_terminal_summary(terminalreporter):
    if not _band_by_test:
        return
    rows = sum(r for r, _ in _band_by_test.values())
    band = sum(b for _, b in _band_by_test.values())
    terminalreporter.write_line(f"near-tie band (ids differ from the oracle's inside 1e-3 of the k-th score): {band} of {rows} selection rows")
    for nodeid, (r, b) in sorted(_band_by_test.items()):
        if b:
            terminalreporter.write_line(f"  {b:5d} of {r:6d} rows  {nodeid}")
