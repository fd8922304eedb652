"""Seeded synthetic input generators shared by the oracle tests, the GPU parity
tests and bench.py.

This module holds NONE of the method's arithmetic (no Gram matrix, no loss, no
solver, no fold construction): it only draws X, y, the lambda grid and the
bandwidth heuristic named by BASELINE.json's `configs`, following the recipe in
SURVEY.md section 8(d) (restated in DESIGN.md "Input recipe").  The paper's own
workloads are a mixture-of-Gaussians simulation and LIBSVM data
sets that are not available offline; these generators stand
in for them with the same shapes (n, p, L, V).

Everything is generated on the host in FP64 with numpy default_rng(seed) and is
handed as the same bytes to the oracle and to the CUDA library.
"""
from __future__ import annotations

import dataclasses
import numpy as np

LOSS_HINGE = 0      # delta-smoothed hinge SVM
LOSS_LOGISTIC = 1   # kernel logistic regression
LOSS_QUANTILE = 2   # kernel quantile regression
LOSS_DWD = 3        # distance-weighted discrimination


@dataclasses.dataclass
class Workload:
    name: str
    X: np.ndarray            # n x p, float64, C-contiguous
    y: np.ndarray            # n, float64 (+-1 for classifiers)
    sigmas: np.ndarray       # bandwidths (lengths), one (K, U) per entry
    lambdas: np.ndarray      # L, descending
    V: int                   # folds
    fold_seed: int
    loss: int
    taus: np.ndarray         # T quantile levels (empty for classifiers)
    smooth0: float           # delta_0 (hinge) or gamma_0 (quantile)
    eta: float               # shrink factor, 0.125
    rounds: int              # R smoothing rounds (1 for logistic)
    m_landmarks: int = 0     # >0: Nystrom with that many landmarks
    landmark_seed: int = 0

    @property
    def n(self):
        return self.X.shape[0]

    @property
    def p(self):
        return self.X.shape[1]

    @property
    def L(self):
        return len(self.lambdas)

    @property
    def T(self):
        return max(1, len(self.taus))

    @property
    def B(self):
        """columns per U: T * L * (V + 1)  (SURVEY.md section 8 notation)."""
        return self.T * self.L * (self.V + 1)


def lambda_grid(hi_exp: float, lo_exp: float, L: int) -> np.ndarray:
    """lambda_l = 10^(hi - l (hi - lo)/(L-1)), l = 0..L-1, descending."""
    if L == 1:
        return np.array([10.0 ** hi_exp])
    l = np.arange(L, dtype=np.float64)
    return 10.0 ** (hi_exp - l * (hi_exp - lo_exp) / (L - 1))


def median_distance(X: np.ndarray, max_rows: int = 5000, seed: int = 12345) -> float:
    """Median Euclidean distance over all pairs of (a seeded subsample of) rows.

    This is the bandwidth heuristic of BASELINE.json ("RBF sigma = median
    pairwise distance"); an input recipe, not part of the method.
    """
    n = X.shape[0]
    if n > max_rows:
        rows = np.random.default_rng(seed).permutation(n)[:max_rows]
        X = X[np.sort(rows)]
        n = max_rows
    from scipy.spatial.distance import pdist
    return float(np.median(pdist(X, metric="euclidean")))


def _flip_labels(y: np.ndarray, frac: float, rng) -> np.ndarray:
    n = len(y)
    k = int(round(frac * n))
    idx = rng.permutation(n)[:k]
    y = y.copy()
    y[idx] = -y[idx]
    return y


def _linear_noisy_labels(n: int, p: int, rng):
    X = rng.standard_normal((n, p))
    beta = rng.standard_normal(p) / np.sqrt(p)
    eps = rng.standard_normal(n)
    s = X @ beta + 0.5 * eps
    y = np.where(s >= 0, 1.0, -1.0)
    y = _flip_labels(y, 0.10, rng)
    return np.ascontiguousarray(X), y


def config0(n: int = 200, p: int = 10, L: int = 20, V: int = 5, seed: int = 1000) -> Workload:
    """Smoothed-hinge SVM, n=200, p=10, 5 folds, 20 lambdas 1e1..1e-4."""
    rng = np.random.default_rng(seed)
    X, y = _linear_noisy_labels(n, p, rng)
    sig = median_distance(X)
    return Workload("cfg0_hinge_n%d_p%d" % (n, p), X, y, np.array([sig]),
                    lambda_grid(1, -4, L), V, 7, LOSS_HINGE, np.zeros(0), 1.0, 0.125, 4)


def config1(n: int = 2000, p: int = 50, L: int = 50, V: int = 5, seed: int = 1001,
            sigma_mults=(0.25, 0.5, 1.0, 2.0, 4.0)) -> Workload:
    """Smoothed-hinge SVM, n=2000, p=50, 5 folds, 50 lambdas 1e2..1e-5 x 5 sigmas."""
    rng = np.random.default_rng(seed)
    X, y = _linear_noisy_labels(n, p, rng)
    sig = median_distance(X)
    return Workload("cfg1_hinge_n%d_p%d" % (n, p), X, y, sig * np.asarray(sigma_mults, dtype=np.float64),
                    lambda_grid(2, -5, L), V, 7, LOSS_HINGE, np.zeros(0), 1.0, 0.125, 4)


def config2(n: int = 10000, p: int = 100, L: int = 100, V: int = 10, seed: int = 1002) -> Workload:
    """Kernel logistic regression, AR(1) features Sigma_ij = 0.5^|i-j|."""
    rng = np.random.default_rng(seed)
    E = rng.standard_normal((n, p))
    X = np.empty((n, p))
    X[:, 0] = E[:, 0]
    for k in range(1, p):
        X[:, k] = 0.5 * X[:, k - 1] + np.sqrt(0.75) * E[:, k]
    beta = rng.standard_normal(p) / np.sqrt(p)
    prob = 1.0 / (1.0 + np.exp(-(X @ beta)))
    y = np.where(rng.random(n) < prob, 1.0, -1.0)
    sig = median_distance(X)
    return Workload("cfg2_logit_n%d_p%d" % (n, p), np.ascontiguousarray(X), y, np.array([sig]),
                    lambda_grid(1, -6, L), V, 7, LOSS_LOGISTIC, np.zeros(0), 0.0, 0.125, 1)


def config3(n: int = 20000, p: int = 28, L: int = 50, V: int = 5, seed: int = 1003,
            taus=(0.1, 0.5, 0.9)) -> Workload:
    """Kernel quantile regression, x~U[-1,1]^p, y = sin(pi sum(x)/sqrt(p)) + t3 noise."""
    rng = np.random.default_rng(seed)
    X = rng.uniform(-1.0, 1.0, size=(n, p))
    y = np.sin(np.pi * X.sum(axis=1) / np.sqrt(p)) + rng.standard_t(3, size=n)
    sig = median_distance(X)
    return Workload("cfg3_kqr_n%d_p%d" % (n, p), np.ascontiguousarray(X), y, np.array([sig]),
                    lambda_grid(1, -6, L), V, 7, LOSS_QUANTILE, np.asarray(taus, dtype=np.float64),
                    1.0, 0.125, 4)


def config4(n: int = 100000, p: int = 50, m: int = 4096, L: int = 100, V: int = 5,
            seed: int = 1004) -> Workload:
    """Nystrom smoothed-hinge SVM, n=100000, p=50, m=4096 landmarks."""
    rng = np.random.default_rng(seed)
    X, y = _linear_noisy_labels(n, p, rng)
    sig = median_distance(X)
    return Workload("cfg4_nys_hinge_n%d_p%d_m%d" % (n, p, m), X, y, np.array([sig]),
                    lambda_grid(2, -6, L), V, 7, LOSS_HINGE, np.zeros(0), 1.0, 0.125, 4,
                    m_landmarks=m, landmark_seed=seed + 17)


def nystrom_paper_shape(name: str) -> Workload:
    """Nystrom workloads with the row and feature counts of the paper's two largest Table-4 data sets
    (covtype 581,012 x 54; MNIST8m 4-vs-6 1,270,178 x 784).  Synthetic rows (the LIBSVM
    files are not in this container), m = 2048 landmarks, 50 lambdas 1e2..1e-5, 5 folds."""
    n, p, seed = {"covtype": (581012, 54, 1044), "mnist8m46": (1270178, 784, 1046)}[name]
    w = config4(n=n, p=p, m=2048, L=50, V=5, seed=seed)
    w.lambdas[:] = lambda_grid(2, -5, 50)
    return w


def landmarks(n: int, m: int, seed: int) -> np.ndarray:
    """m distinct row indices: first m entries of a seeded permutation."""
    return np.sort(np.random.default_rng(seed).permutation(n)[:m]).astype(np.int64)


def new_points(w: Workload, n_new: int, seed: int = 99) -> np.ndarray:
    """Fresh rows from (roughly) the training distribution, for tkm_predict tests."""
    rng = np.random.default_rng(seed)
    idx = rng.integers(0, w.n, size=n_new)
    return np.ascontiguousarray(w.X[idx] + 0.3 * rng.standard_normal((n_new, w.p)) * w.X.std())


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}
