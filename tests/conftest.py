import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture
def knobs():
    """Typed debug knobs of the library (bt_debug_knob): knobs(name, value); everything back to the default afterwards."""
    import paper_2208_02382_b200 as bt
    touched = []

    def set_knob(name, value):
        bt.debug_knob(name, int(value))
        touched.append(name)

    yield set_knob
    for name in touched:
        bt.debug_knob(name, -1)
