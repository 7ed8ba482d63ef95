import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def orc():
    from oracle import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session")
def dense44(orc):
    """Config-0 lattice (4^4, U = exp(0.3 i H)): dense K from the oracle, its eigendecomposition."""
    from paper_1510_06897_b200 import inputs
    dims = (4, 4, 4, 4)
    U = inputs.random_links(dims, 0.3, inputs.SEED_BASE + 0)
    K = orc.dense_k(dims, U)
    S, lam, W = orc.exact_sign_dense(K)
    return dict(dims=dims, U=U, K=K, S=S, lam=lam, W=W)


def rel_err(a, b):
    a = np.asarray(a)
    b = np.asarray(b)
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))
