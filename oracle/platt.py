"""Oracle: Platt scaling of decision values into class probabilities (test infrastructure).

PAPER.md:49, 73-74, 79 (`probability=True`, `predict_proba`) and 250-256 (section A.7) say only that a
sigmoid is fitted to the raw decision scores; the construction is not printed.  Reading G21:
Platt's method as specified by Lin, Lin and Weng (2007): with N+ / N- the class counts and targets
t+ = (N+ + 1)/(N+ + 2), t- = 1/(N- + 2),

    (A, B) = argmin  - sum_i [ t_i log p_i + (1 - t_i) log(1 - p_i) ],   p_i = 1 / (1 + exp(A f_i + B)),

a strictly convex problem in (A, B) for non-degenerate scores, solved here by a damped Newton iteration
with backtracking from (0, log((N- + 1)/(N+ + 1))).  The scores are the HELD-OUT decision values of the
exact cross-validation at the selected lambda, which the path produces without refitting.

Pins (tests/test_oracle_platt.py): gradient zero at the solution; agreement with scikit-learn's independent
implementation of the same method; invariance of p under the (A, B) of shifted/scaled scores.
"""
import numpy as np


def platt_targets(y):
    y = np.asarray(y, dtype=np.float64)
    n_pos = float(np.sum(y > 0))
    n_neg = float(len(y) - n_pos)
    t = np.where(y > 0, (n_pos + 1.0) / (n_pos + 2.0), 1.0 / (n_neg + 2.0))
    return t, n_pos, n_neg


def platt_objective(f, t, A, B):
    """- sum t log p + (1 - t) log(1 - p), overflow-safe (Lin, Lin & Weng eq. for fApB >= 0 / < 0)."""
    s = A * f + B
    return float(np.sum(np.where(s >= 0, t * s + np.log1p(np.exp(-np.abs(s))),
                                 (t - 1.0) * s + np.log1p(np.exp(-np.abs(s))))))


def platt_fit(f, y, maxit=100, min_step=1e-10, sigma=1e-12, eps=1e-5):
    """Returns (A, B).  Newton with backtracking exactly as in Lin, Lin & Weng (2007), Algorithm 1."""
    f = np.asarray(f, dtype=np.float64)
    t, n_pos, n_neg = platt_targets(y)
    A, B = 0.0, float(np.log((n_neg + 1.0) / (n_pos + 1.0)))
    fval = platt_objective(f, t, A, B)
    for _ in range(maxit):
        s = A * f + B
        e = np.exp(-np.abs(s))
        p = np.where(s >= 0, e / (1.0 + e), 1.0 / (1.0 + e))      # p_i = 1/(1 + exp(s_i))
        q = 1.0 - p
        d2 = p * q
        h11 = sigma + float(np.sum(f * f * d2))
        h22 = sigma + float(np.sum(d2))
        h21 = float(np.sum(f * d2))
        d1 = t - p
        g1 = float(np.sum(f * d1))
        g2 = float(np.sum(d1))
        if abs(g1) < eps and abs(g2) < eps:
            break
        det = h11 * h22 - h21 * h21
        dA = -(h22 * g1 - h21 * g2) / det
        dB = -(-h21 * g1 + h11 * g2) / det
        gd = g1 * dA + g2 * dB
        step = 1.0
        while step >= min_step:
            nA, nB = A + step * dA, B + step * dB
            nf = platt_objective(f, t, nA, nB)
            if nf < fval + 1e-4 * step * gd:
                A, B, fval = nA, nB, nf
                break
            step /= 2.0
        if step < min_step:
            break
    return A, B


def platt_proba(f, A, B):
    s = A * np.asarray(f, dtype=np.float64) + B
    e = np.exp(-np.abs(s))
    return np.where(s >= 0, e / (1.0 + e), 1.0 / (1.0 + e))


def cv_decision_values(spec, res, foldid, t, l, L, V):
    """Held-out decision value of every row at (t, lambda_l): row j is scored by the column that held out
    fold foldid[j] (the masked fit restricted to the training rows is the refit)."""
    n = spec.n
    f = np.empty(n)
    for v in range(V):
        c = (t * (V + 1) + v) * L + l
        rows = np.nonzero(np.asarray(foldid) == v)[0]
        f[rows] = spec.U[rows] @ (spec.lam * res.a[:, c]) + res.beta0[c]
    return f
