import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def oracle_mod():
    from oracle import tso
    tso.build()
    return tso


class SimpleCam:
    def __init__(self, width, height, fx, fy, cx, cy, znear=0.2):
        self.width, self.height, self.fx, self.fy, self.cx, self.cy, self.znear = width, height, fx, fy, cx, cy, znear


class SimpleParams:
    def __init__(self, sigma=1.0, alpha_min=0.0, t_min=0.0, eps_area=1e-6, lambda_dep=0.05, min_opacity=False,
                 tight_binning=False):
        self.sigma, self.alpha_min, self.t_min, self.eps_area, self.lambda_dep = sigma, alpha_min, t_min, eps_area, lambda_dep
        self.min_opacity, self.tight_binning = min_opacity, tight_binning


IDENT = np.concatenate([np.eye(3), np.zeros((3, 1))], axis=1)


def unproject(uvz, cam):
    """World points (identity pose) that project exactly to pixel (u,v) at depth z -- test-side helper."""
    uvz = np.asarray(uvz, dtype=np.float64)
    X = (uvz[:, 0] - cam.cx) / cam.fx * uvz[:, 2]
    Y = (uvz[:, 1] - cam.cy) / cam.fy * uvz[:, 2]
    return np.stack([X, Y, uvz[:, 2]], axis=1)
