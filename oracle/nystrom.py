"""Nystrom spectral setup (test infrastructure).  PAPER.md:242 says only that ONE Nystrom
approximation of K is built outside the lambda-path and CV loops; reading G11 (SURVEY.md
8(c)) fixes the construction:

  landmarks idx (m distinct rows);  K_mm = W Theta W^T, drop Theta_i <= 1e-12 Theta_max;
  Phi = K_nm W Theta^-1/2  (n x r');  Phi^T Phi = Q Lam Q^T, drop Lam_i <= 1e-12 Lam_max;
  thin U = Phi Q Lam^-1/2  (n x r, orthonormal columns);  K~ = Phi Phi^T = U Lam U^T.
  Landmark weights: gamma = W Theta^-1/2 Q Lam^1/2 a, so f(x) = sum_l k(x, x_l) gamma_l + b0.
"""
import numpy as np

from .gram import gram_rbf
from .spectral import Spectral

RANK_TOL = 1e-12


def nystrom_setup(X, sigma, landmark_idx):
    X = np.asarray(X, dtype=np.float64)
    idx = np.asarray(landmark_idx, dtype=np.int64)
    n = X.shape[0]
    K_nm = gram_rbf(X, sigma, X[idx])
    K_mm = gram_rbf(X[idx], sigma)
    theta, W = np.linalg.eigh(K_mm)
    keep = theta > RANK_TOL * theta.max()
    theta, W = theta[keep], W[:, keep]
    Wt = W / np.sqrt(theta)[None, :]                 # W Theta^-1/2, m x r'
    Phi = K_nm @ Wt                                  # n x r'
    lam, Q = np.linalg.eigh(Phi.T @ Phi)
    keep2 = lam > RANK_TOL * lam.max()
    lam, Q = lam[keep2], Q[:, keep2]
    U = (Phi @ Q) / np.sqrt(lam)[None, :]            # n x r
    u1 = U.T @ np.ones(n)
    lmap = Wt @ (Q * np.sqrt(lam)[None, :])          # m x r
    return Spectral(U=U, lam=lam, u1=u1, n=n, r=U.shape[1], landmark_map=lmap, landmark_idx=idx)


def nystrom_landmark_weights(spec, a):
    """gamma (m) from spectral coordinates a (r)."""
    return spec.landmark_map @ a
