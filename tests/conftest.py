import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def theta0():
    import numpy as np
    # fiducial truth of SURVEY.md section 8(d): H0, Om, alpha, beta, mmin, mmax, mu, sigma, lambda, gamma, kappa, zp
    return np.array([70.0, 0.3, 3.4, 1.1, 5.0, 100.0, 35.0, 4.0, 0.04, 2.7, 2.9, 1.9])
