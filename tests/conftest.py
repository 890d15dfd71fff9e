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
    """The fp64 CPU oracle (oracle/md_oracle.c), built on demand."""
    from oracle import md_oracle
    md_oracle.build()
    return md_oracle


@pytest.fixture(autouse=True)
def _oracle_parameters_do_not_leak():
    """The oracle's C library takes the parameters of kinds 2-5 (and the thermostat chain length) as a call
    argument; its Python wrapper passes a default Params object that the set_* functions fill.  Every test
    starts with that object in the UNSET state, so none can pass on what another left behind."""
    from oracle import md_oracle
    if os.path.exists(md_oracle._LIB):
        md_oracle.reset_params()
    yield


@pytest.fixture(scope="session")
def W():
    from paper_1912_04232_b200 import workloads
    return workloads


def golden(name):
    """Parse tests/golden/<name>: 'key = value' lines, '#' comments."""
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            k, v = line.split("=", 1)
            out[k.strip()] = float(v)
    return out
