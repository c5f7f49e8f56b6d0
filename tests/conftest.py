import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200, sm_100a); run with -m gpu")


@pytest.fixture(scope="session")
def tiny_case():
    """BASELINE.json configs[0]: M=16, K=256, N=256, 64x64 blocks, top-2 of 16, seed 0.
    X_cal = the fp32 image of A itself (16 tokens), DESIGN.md input recipe."""
    import numpy as np
    import oracle
    import synth

    W = synth.gen_weight(0, 256, 256)
    A = synth.gen_act(0, 16, 256, n_outlier_ch=2)
    h = oracle.hessian_diag(A.astype(np.float32)).astype(np.float32)
    L = oracle.algorithm1(W, h, 64, 2)
    return dict(W=W, A=A, h=h, L=L)
