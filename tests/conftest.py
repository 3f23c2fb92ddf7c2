import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def make_obs(mod, d):
    """Build a library-specific observable struct from a plain coefficient dict (chfpe_inputs.observable)."""
    return mod.make_observable(d["c0"], d["lin_q"], d["quad"], d["lin_p"])
