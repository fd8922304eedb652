"""Oracle step O3: loss table (test infrastructure).

psi(y, f) = d loss / d f, curvature = sup loss'' (= 1/kappa),
nominal loss = the non-smoothed loss used to score cross-validation.

  smoothed hinge   PAPER.md:138 (L_delta), kappa = 2 delta
  logistic         not printed: reading G9, log(1 + exp(-y f)), curv 1/4
  DWD              not printed (PAPER.md:47, 81, 85 name the estimator; it cites Wang and Zou 2018): reading
                   G20, the generalised DWD loss with q = 1,  V(u) = 1 - u (u <= 1/2), 1/(4u) (u > 1/2),
                   which is C^1 with sup V'' = V''(1/2+) = 4; no smoothing round
  smoothed check   not printed: reading G10, the C^1 quadratic blend of the
                   check loss rho_tau on [-gamma, gamma], curvature 1/(2 gamma)
"""
import numpy as np

LOSS_HINGE = 0
LOSS_LOGISTIC = 1
LOSS_QUANTILE = 2
LOSS_DWD = 3


def curvature(loss, smooth):
    """sup of the second derivative in f (the paper's 1/kappa)."""
    if loss == LOSS_HINGE:
        return 1.0 / (2.0 * smooth)          # kappa = 2 delta
    if loss == LOSS_LOGISTIC:
        return 0.25
    if loss == LOSS_QUANTILE:
        return 1.0 / (2.0 * smooth)
    if loss == LOSS_DWD:
        return 4.0                           # V''(u) = 1/(2 u^3) on u > 1/2, largest at u = 1/2
    raise ValueError(loss)


def psi(loss, y, f, smooth=None, tau=None):
    """d loss(y, f) / d f, elementwise; y and f broadcast."""
    y = np.asarray(y, dtype=np.float64)
    f = np.asarray(f, dtype=np.float64)
    if loss == LOSS_HINGE:
        d = smooth
        u = y * f
        # L'_delta(u): -1 | (u - 1 - delta)/(2 delta) | 0
        lp = np.where(u <= 1.0 - d, -1.0, np.where(u >= 1.0 + d, 0.0, (u - 1.0 - d) / (2.0 * d)))
        return y * lp
    if loss == LOSS_LOGISTIC:
        u = y * f
        # -y / (1 + e^u), written to avoid overflow for large |u|
        e = np.exp(-np.abs(u))
        sig_neg = np.where(u >= 0, e / (1.0 + e), 1.0 / (1.0 + e))   # = 1/(1+e^u)
        return -y * sig_neg
    if loss == LOSS_QUANTILE:
        g = smooth
        t = y - f
        hp = np.where(t < -g, tau - 1.0, np.where(t > g, tau, t / (2.0 * g) + tau - 0.5))
        return -hp
    if loss == LOSS_DWD:
        u = y * f
        us = np.maximum(u, 0.5)               # keeps the unused branch finite
        return y * np.where(u <= 0.5, -1.0, -1.0 / (4.0 * us * us))
    raise ValueError(loss)


def smooth_loss(loss, y, f, smooth=None, tau=None):
    """The smoothed loss itself (objective values for the descent / refit pins)."""
    y = np.asarray(y, dtype=np.float64)
    f = np.asarray(f, dtype=np.float64)
    if loss == LOSS_HINGE:
        d = smooth
        u = y * f
        return np.where(u <= 1.0 - d, 1.0 - u,
                        np.where(u >= 1.0 + d, 0.0, (u - (1.0 + d)) ** 2 / (4.0 * d)))
    if loss == LOSS_LOGISTIC:
        u = y * f
        return np.maximum(-u, 0.0) + np.log1p(np.exp(-np.abs(u)))
    if loss == LOSS_QUANTILE:
        g = smooth
        t = y - f
        return np.where(t < -g, (tau - 1.0) * t,
                        np.where(t > g, tau * t, t * t / (4.0 * g) + t * (tau - 0.5) + g / 4.0))
    if loss == LOSS_DWD:
        u = y * f
        return np.where(u <= 0.5, 1.0 - u, 1.0 / (4.0 * np.maximum(u, 0.5)))
    raise ValueError(loss)


def nominal_loss(loss, y, f, tau=None):
    """Non-smoothed loss for CV scoring: hinge, deviance, check loss."""
    y = np.asarray(y, dtype=np.float64)
    f = np.asarray(f, dtype=np.float64)
    if loss == LOSS_HINGE:
        return np.maximum(1.0 - y * f, 0.0)
    if loss == LOSS_LOGISTIC:
        u = y * f
        return np.maximum(-u, 0.0) + np.log1p(np.exp(-np.abs(u)))
    if loss == LOSS_QUANTILE:
        t = y - f
        return t * (tau - (t < 0))
    if loss == LOSS_DWD:
        u = y * f
        return np.where(u <= 0.5, 1.0 - u, 1.0 / (4.0 * np.maximum(u, 0.5)))
    raise ValueError(loss)
