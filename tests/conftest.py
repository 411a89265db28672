import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


@pytest.fixture(scope="session")
def tiny_dims():
    from pf_synth import Dims
    return Dims(c_m=8, c_z=8, heads_msa=2, heads_pair=2, head_dim=4, c_opm=3, c_tri=5, transition_n=2)
