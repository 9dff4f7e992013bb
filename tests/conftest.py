import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def cfg0():
    from synth import workloads
    return workloads.make(0)


@pytest.fixture(scope="session")
def cfg0_oracle(cfg0):
    from oracle import oracle as orc
    av = orc.avatar_load(cfg0)
    return av, orc.render_frame(av, cfg0, vis_mode=0), orc.render_frame(av, cfg0, vis_mode=1)
