import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def tiny_problem():
    """n=60 hinge problem shared by several oracle pins (K, spectral, folds)."""
    import numpy as np
    import oracle as o
    import workloads as wl
    w = wl.config0(n=60, p=5, L=3, V=4, seed=11)
    K = o.gram_rbf(w.X, w.sigmas[0])
    spec = o.spectral_setup(K)
    foldid = o.make_folds(w.n, w.V, w.fold_seed)
    return dict(w=w, K=K, spec=spec, foldid=foldid, np=np)
