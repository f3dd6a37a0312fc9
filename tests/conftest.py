import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def cfg1():
    """Config 1 with its oracle-tabulated G, weights, lambda and noisy data (shared by several pins)."""
    import numpy as np
    import oracle
    from paper_2602_03857_b200 import workloads
    wl = workloads.make(1)
    mesh = oracle.Mesh(wl.xn, wl.yn, wl.zn)
    G = oracle.tabulate(mesh, wl.xo, wl.yo, wl.zo, wl.gamma)
    w = oracle.depth_weights(mesh, wl.beta, wl.z0)
    diag = oracle.gram_diag(G, w)
    lam = wl.lam_factor * diag.sum() / wl.N
    d_clean = oracle.dense_matvec(G, wl.m_true)
    sigma = wl.noise_frac * np.abs(d_clean).max()
    d_obs = d_clean + sigma * wl.noise()
    return dict(wl=wl, mesh=mesh, G=G, w=w, diag=diag, lam=lam, d_clean=d_clean, d_obs=d_obs)
