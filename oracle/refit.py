"""Definitions the pins compare against (test infrastructure): the objective (1), the dense
bordered majoriser, and the brute-force per-fold refit that exact CV avoids.

PAPER.md:126 eq. (1); PAPER.md:146/176 (H_lambda) with the intercept border of reading G2;
PAPER.md:160-162 (the refit on K_[v], the (n-m) x (n-m) sub-kernel).
"""
import numpy as np

from .losses import smooth_loss, nominal_loss
from .spectral import spectral_setup
from .path import fit_column


def objective(K, y, alpha, beta0, lam, loss, mask=None, smooth=None, tau=None, nominal=False):
    """(1/n_c) sum_j M_j loss(y_j, K_j^T alpha + beta0) + lam alpha^T K alpha."""
    n = K.shape[0]
    mask = np.ones(n) if mask is None else mask
    f = K @ alpha + beta0
    lv = nominal_loss(loss, y, f, tau) if nominal else smooth_loss(loss, y, f, smooth, tau)
    return float(np.sum(mask * lv) / mask.sum() + lam * alpha @ K @ alpha)


def dense_majoriser(K, lam, c):
    """P = [[c n, c 1^T K], [c K 1, 2 lam K + c K K]]  ((n+1) x (n+1)), reading G1/G2."""
    n = K.shape[0]
    one = np.ones(n)
    P = np.empty((n + 1, n + 1))
    P[0, 0] = c * n
    P[0, 1:] = c * (one @ K)
    P[1:, 0] = c * (K @ one)
    P[1:, 1:] = 2.0 * lam * K + c * (K @ K)
    return P


def brute_force_refit(K, y, foldid, v, lam, loss, levels, tau=None, tol=1e-12, maxit=200000):
    """Refit on the training rows alone: own eigendecomposition of K[act, act], all-ones
    mask, divisor n - m.  Returns (act, alpha_act, beta0, f_heldout, rows_v)."""
    foldid = np.asarray(foldid)
    act = np.nonzero(foldid != v)[0]
    rows = np.nonzero(foldid == v)[0]
    Ka = K[np.ix_(act, act)]
    spec = spectral_setup(Ka)
    a, b0, it, kkt, flag = fit_column(spec, y[act], loss, levels, lam, np.ones(len(act)),
                                      tau=tau, tol=tol, maxit=maxit)
    alpha = spec.U @ a
    f_out = K[np.ix_(rows, act)] @ alpha + b0
    return act, alpha, b0, f_out, rows
