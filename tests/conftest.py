import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import ns_oracle
    return ns_oracle


@pytest.fixture(scope="session")
def k53_512():
    """BASELINE.json configs[4] input (512^3 Gaussian k^-5/3 field, seed 5): 40 s of numpy FFTs, shared by the full-size tests."""
    from paper_2401_09843_b200 import inputs
    return inputs.gaussian_k53(512, seed=5)


@pytest.fixture(scope="session")
def k53_512_hat(k53_512):
    """The spectral state of k53_512 by the numpy restatement of set_initial (tests/_sampling.py): the common input of the CUDA
    path and the oracle at 512^3 -- no oracle input comes from the CUDA path."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from _sampling import spectral_state
    return spectral_state(k53_512)


@pytest.fixture(scope="session")
def oracle2d():
    from oracle import ns2d_oracle
    return ns2d_oracle
