import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def cfg2_oracle_cloud():
    """Oracle cloud of BASELINE.json configs[1] (monodisperse 5 um, 2 mg/cm^2), built once."""
    import pdv_workloads as W
    from oracle import cloud
    return cloud.build_cloud(W.config(1)["clouds"][0])


@pytest.fixture(scope="session")
def _library_is_built():
    """The in-tree CUDA library is (re)built once per session when a source is newer than it (nvcc cross-compiles without a
    GPU).  Requested only by the modules that load the library (ABI, shard, GPU tests: `pytestmark = usefixtures(...)`); the
    oracle's own pins (tests/test_oracle_*.py) neither build nor load the product, so they run on a box without nvcc and an
    nvcc failure cannot mask an oracle failure."""
    from paper_2012_00963_b200 import build as pbuild
    pbuild.build()
