"""Oracle steps O7-O8: exact cross-validation scores and prediction (test infrastructure).

PAPER.md:160-168 (exact CV formula: the masked full-size fit, restricted to the training
rows, IS the refit on those rows), PAPER.md:238 (V-fold: "fold-wise validation loss
values" from the same spectral quantities), PAPER.md:72 (predict).
Readings: G14 (select on pooled mean nominal loss; ties -> largest lambda), G15
(label(0) = +1).
"""
import numpy as np

from .gram import gram_rbf
from .losses import nominal_loss, LOSS_QUANTILE


def label_of(f):
    """+1 if f >= 0 else -1, int8 (G15)."""
    return np.where(np.asarray(f) >= 0.0, 1, -1).astype(np.int8)


def exact_cv(spec, res, y, foldid, loss, taus=()):
    """Returns cv_loss[T, L, V], cv_err[T, L, V] (int64; -1 for regression),
    cv_mean[T, L], best_l[T].

    For column (t, l, v), v < V:  f_j = [U (Lam * a_c)]_j + b0_c on the rows j of fold v;
    cv_loss = mean nominal loss over those rows; cv_err = #{label(f_j) != y_j};
    cv_mean[t, l] = (1/n) sum_v |v| cv_loss[t, l, v];  best_l = argmin_l cv_mean, ties ->
    the largest lambda.
    """
    cols = res.cols
    L, V, T = cols["L"], cols["V"], cols["T"]
    y = np.asarray(y, dtype=np.float64)
    foldid = np.asarray(foldid)
    n = len(y)
    lambdas = np.empty(L)
    cv_loss = np.zeros((T, L, V))
    cv_err = np.full((T, L, V), -1, dtype=np.int64)
    for t in range(T):
        tau = float(taus[t]) if loss == LOSS_QUANTILE else None
        for v in range(V):
            rows = np.nonzero(foldid == v)[0]
            for l in range(L):
                c = (t * (V + 1) + v) * L + l
                lambdas[l] = cols["lam"][c]
                f = spec.U[rows] @ (spec.lam * res.a[:, c]) + res.beta0[c]
                cv_loss[t, l, v] = float(np.mean(nominal_loss(loss, y[rows], f, tau)))
                if loss != LOSS_QUANTILE:
                    cv_err[t, l, v] = int(np.sum(label_of(f) != y[rows].astype(np.int8)))
    sizes = np.array([np.sum(foldid == v) for v in range(V)], dtype=np.float64)
    cv_mean = (cv_loss * sizes[None, None, :]).sum(axis=2) / n
    best_l = np.zeros(T, dtype=np.int64)
    for t in range(T):
        best, bl = np.inf, 0
        for l in range(L):
            m = cv_mean[t, l]
            if m < best or (m == best and lambdas[l] > lambdas[bl]):
                best, bl = m, l
        best_l[t] = bl
    return cv_loss, cv_err, cv_mean, best_l


def predict(X_train, alpha, beta0, sigma, X_new):
    """f(x) = sum_i exp(-||x - x_i||^2 / (2 sigma^2)) alpha_i + beta0; labels by label_of.
    For Nystrom pass the landmark rows as X_train and the landmark weights as alpha."""
    Kx = gram_rbf(X_new, sigma, X_train)
    f = Kx @ np.asarray(alpha, dtype=np.float64) + beta0
    return f, label_of(f)
