"""Oracle step O1: RBF Gram matrix (test infrastructure; see oracle/__init__.py).

PAPER.md:69 names kernel="rbf" and never prints the formula; reading G12
(SURVEY.md 8(c)): k(x, x') = exp(-||x - x'||^2 / (2 sigma^2)), sigma a length.
"""
import numpy as np


def gram_rbf(X, sigma, X2=None):
    """K[i, j] = exp(-sum_k (X[i,k] - X2[j,k])^2 / (2 sigma^2)), direct differences, FP64.

    X: n x p, X2: n2 x p (None => X).  Returns n x n2 float64.
    The definition written out: no norm expansion, no blocking beyond a row loop.
    """
    X = np.asarray(X, dtype=np.float64)
    Y = X if X2 is None else np.asarray(X2, dtype=np.float64)
    if not sigma > 0:
        raise ValueError("sigma must be > 0")
    n, n2 = X.shape[0], Y.shape[0]
    K = np.empty((n, n2), dtype=np.float64)
    inv = 1.0 / (2.0 * sigma * sigma)
    for i in range(n):
        d = Y - X[i]                      # n2 x p differences
        d2 = np.einsum("jk,jk->j", d, d)  # squared distances
        K[i] = np.exp(-d2 * inv)
    return K
