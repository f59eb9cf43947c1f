import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def cfg1():
    from paper_2601_19714_b200 import synth
    return synth.make_config(1)


@pytest.fixture(scope="session")
def cfg1_oracle(cfg1):
    import oracle
    wl = cfg1
    return oracle.image(wl.uvw_m, wl.freq_hz, wl.vis, wl.weights, wl.n, wl.n_wplanes, wl.support,
                        wl.pixel_rad, want_stacks=True, want_raw=True)
