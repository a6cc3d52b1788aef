import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: long-running parity case")


def pytest_terminal_summary(terminalreporter):
    try:
        import parity_helpers
        if parity_helpers.WORST_R["frac"] > 0:
            terminalreporter.write_line(f"largest logged-ratio error of the session: {parity_helpers.WORST_R['frac']:.3e} of the tolerance "
                                        f"(rtol {parity_helpers.R_RTOL:g}, atol {parity_helpers.R_ATOL:g})")
    except Exception:
        pass
