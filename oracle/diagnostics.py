"""Oracle: duality-gap certificate of a path column for the NON-smoothed problem (test infrastructure).

PAPER.md:220-222 (Alg. 1 l.22-24) shrinks delta "until the KKT conditions of all SVM models are satisfied" but
prints neither the test nor its tolerance; reading G7 keeps a fixed delta-schedule and REPORTS the violation as
a diagnostic.  The diagnostic is the duality gap of the original problem (reading G22):

  primal  P(alpha, beta0) = (1/n_c) sum_{j in train} loss(y_j, f_j) + lam alpha^T K alpha,   f = K alpha + beta0
          with the nominal loss: hinge max(0, 1 - y f) or the check loss rho_tau(y - f);
  dual    hinge     : loss = max_{theta in [0,1]} theta (1 - y f)   =>  D(theta) = (1/n_c) sum theta_j - lam alpha^T K alpha
          check loss: loss = max_{s in [tau-1,tau]} s (y - f)       =>  D(s)     = (1/n_c) sum s_j y_j - lam alpha^T K alpha
          both under  sum_j y_j theta_j = 0 (resp. sum_j s_j = 0)  and  alpha = -z / (2 lam)  with
          z_j = -y_j theta_j / n_c (resp. -s_j / n_c) on the training rows, 0 on the held-out rows.

A solution of the smoothed problem supplies a dual-feasible point for free: z_j = psi_delta(y_j, f_j) / n_c has
theta_j = -L'_delta(y_j f_j) in [0, 1] (s_j = H'_gamma(y_j - f_j) in [tau-1, tau]), and the smoothed stationarity
conditions (P6) are exactly the two dual constraints.  Hence  0 <= P - P* <= gap = P - D,  which goes to zero with
delta.  Written out in the alpha domain; nothing here is shared with the CUDA path.

Pins (tests/test_oracle_diagnostics.py): gap >= 0; gap = O(delta) and shrinks with the smoothing level; weak
duality D <= P(any other primal point); D <= P* <= P with P* from scikit-learn's SVC dual solver.
"""
import numpy as np

from .losses import LOSS_HINGE, LOSS_QUANTILE, nominal_loss, psi


def duality_gap(spec, res, y, loss):
    """Per column c of a PathResult: (P_c, D_c, gap_c) of the non-smoothed problem at (alpha_c, beta0_c)."""
    if loss not in (LOSS_HINGE, LOSS_QUANTILE):
        raise ValueError("the duality-gap diagnostic is defined for the smoothed (hinge, check) losses")
    y = np.asarray(y, dtype=np.float64)
    cols = res.cols
    B = cols["B"]
    P, D = np.empty(B), np.empty(B)
    for c in range(B):
        a = res.a[:, c]
        f = spec.U @ (spec.lam * a) + res.beta0[c]          # K alpha + beta0 with alpha = U a
        quad = float(np.sum(spec.lam * a * a))               # alpha^T K alpha
        M, nc, lam = cols["M"][:, c], cols["n_c"][c], cols["lam"][c]
        tau = None if np.isnan(cols["tau"][c]) else float(cols["tau"][c])
        P[c] = float(np.sum(M * nominal_loss(loss, y, f, tau))) / nc + lam * quad
        smooth = res.smooth_final if res.smooth_col is None else float(res.smooth_col[c])   # the column's own level (G23)
        dual_var = -psi(loss, y, f, smooth, tau)             # hinge: y_j theta_j ; check loss: s_j
        D[c] = float(np.sum(M * dual_var * y)) / nc - lam * quad
    return P, D, P - D
