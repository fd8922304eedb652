"""Oracle step O2: one-time eigendecomposition K = U Lam U^T (test infrastructure).

PAPER.md:184 (Algorithm 1 line 3).  Eigenvalues are clamped to
>= 0 only (reading G16): only Lam Pi^-1 = 1/(2 lam + c Lam) ever appears
(PAPER.md:187, 207), which is finite at Lam = 0.
"""
import dataclasses
import numpy as np


@dataclasses.dataclass
class Spectral:
    U: np.ndarray      # n x r   (r = n full kernel; r <= m Nystrom)
    lam: np.ndarray    # r eigenvalues, >= 0
    u1: np.ndarray     # r, U^T 1
    n: int
    r: int
    # Nystrom only (None for the full kernel): map spectral coords -> landmark weights
    landmark_map: np.ndarray = None   # m x r, gamma = landmark_map @ a
    landmark_idx: np.ndarray = None


def spectral_setup(K):
    """Lam, U = eigh(K) in FP64 (LAPACK); Lam <- max(Lam, 0); u1 = U^T 1."""
    K = np.asarray(K, dtype=np.float64)
    n = K.shape[0]
    lam, U = np.linalg.eigh(K)
    lam = np.maximum(lam, 0.0)
    u1 = U.T @ np.ones(n)
    return Spectral(U=U, lam=lam, u1=u1, n=n, r=n)
