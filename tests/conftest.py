import os
import sys
import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def mlp2():
    import synth
    return synth.xavier_mlp(synth.MLP2_DIMS, 1)


@pytest.fixture(scope="session")
def mlp2_bias():
    import synth
    return synth.xavier_mlp(synth.MLP2_DIMS, 1, bias_scale=0.3)


@pytest.fixture(scope="session")
def mlp3():
    import synth
    return synth.xavier_mlp(synth.MLP3_DIMS, 3)


def zero_mlp(dims, b_last=None):
    Ws = [np.zeros((dims[l + 1], dims[l]), np.float32) for l in range(len(dims) - 1)]
    bs = [np.zeros(dims[l + 1], np.float32) for l in range(len(dims) - 1)]
    if b_last is not None:
        bs[-1][:] = np.asarray(b_last, np.float32)
    return Ws, bs


def rel_l2(a, b):
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))
