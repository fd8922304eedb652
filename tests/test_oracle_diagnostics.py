"""Pins of oracle.duality_gap (P17; reading G22): the certificate must be non-negative, O(delta), shrink with the
smoothing level, obey weak duality against arbitrary primal points, and bracket the optimum of an independent
solver (scikit-learn's SVC on the same precomputed kernel)."""
import numpy as np
import pytest

import oracle as o
import workloads as wl
from oracle import LOSS_HINGE, LOSS_QUANTILE


def _hinge_problem(n=80, seed=33):
    w = wl.config0(n=n, p=4, seed=seed)
    K = o.gram_rbf(w.X, wl.median_distance(w.X))
    return w.X, w.y, K, o.spectral_setup(K)


def test_gap_is_nonnegative_order_delta_and_shrinks_with_the_smoothing_level():
    n, V = 72, 3
    X, y, K, spec = _hinge_problem(n)
    foldid = o.make_folds(n, V, 9)
    lambdas = np.array([1e-1, 1e-2, 1e-3])
    prev = None
    for rounds in (2, 3, 4):
        res = o.fit_path(spec, y, LOSS_HINGE, lambdas, foldid, V, rounds=rounds, tol=1e-12, maxit=400000)
        P, D, gap = o.duality_gap(spec, res, y, LOSS_HINGE)
        delta = res.smooth_final
        assert np.all(gap >= -1e-10)
        assert np.all(gap <= delta)                       # zone rows: hinge - theta (1 - u) <= delta / 4 each, and
        if prev is not None:                              # the quadratic terms cancel at stationarity
            assert np.all(gap <= prev * 0.5 + 1e-9)       # eta = 1/8 per round: at least halves
        prev = gap
    assert prev.max() < 1e-3


def test_weak_duality_against_other_primal_points():
    n = 60
    X, y, K, spec = _hinge_problem(n, seed=5)
    foldid = o.make_folds(n, 3, 2)
    lambdas = np.array([3e-2, 1e-3])
    res = o.fit_path(spec, y, LOSS_HINGE, lambdas, foldid, 3, rounds=3, tol=1e-12, maxit=400000)
    P, D, gap = o.duality_gap(spec, res, y, LOSS_HINGE)
    rng = np.random.default_rng(0)
    for c in range(res.cols["B"]):
        M, lam = res.cols["M"][:, c], res.cols["lam"][c]
        alpha_c, b_c = o.path_coef(spec, res, c)
        # the column's own primal value, recomputed in the alpha domain by the refit module's objective
        assert P[c] == pytest.approx(o.objective(K, y, alpha_c, b_c, lam, LOSS_HINGE, mask=M, nominal=True), rel=1e-12)
        for scale in (1e-3, 1e-1, 1.0):
            alpha = alpha_c + scale * rng.standard_normal(n) * np.abs(alpha_c).max()
            b = b_c + scale * rng.standard_normal()
            assert o.objective(K, y, alpha, b, lam, LOSS_HINGE, mask=M, nominal=True) >= D[c] - 1e-10


def test_gap_brackets_the_svc_optimum():
    from sklearn.svm import SVC
    n = 80
    X, y, K, spec = _hinge_problem(n)
    foldid = np.zeros(n, dtype=np.int64)
    foldid[::2] = 1                                        # V = 2; the v = V column is the full-data fit
    for lam in (1e-2, 1e-3):
        svc = SVC(C=1.0 / (2 * n * lam), kernel="precomputed", tol=1e-10).fit(K, y)
        alpha_qp = np.zeros(n)
        alpha_qp[svc.support_] = svc.dual_coef_[0]
        p_star = o.objective(K, y, alpha_qp, float(svc.intercept_[0]), lam, LOSS_HINGE, nominal=True)
        res = o.fit_path(spec, y, LOSS_HINGE, np.array([lam]), foldid, 2, rounds=4, tol=1e-12, maxit=400000)
        P, D, gap = o.duality_gap(spec, res, y, LOSS_HINGE)
        c = 2                                              # (t = 0, v = V = 2, l = 0)
        assert D[c] - 1e-8 <= p_star <= P[c] + 1e-8
        assert gap[c] <= res.smooth_final


def test_check_loss_gap():
    n = 64
    rng = np.random.default_rng(3)
    X = rng.uniform(-1, 1, (n, 3))
    y = np.sin(np.pi * X.sum(1)) + 0.3 * rng.standard_t(3, n)
    K = o.gram_rbf(X, wl.median_distance(X))
    spec = o.spectral_setup(K)
    foldid = o.make_folds(n, 4, 1)
    taus = (0.2, 0.8)
    res = o.fit_path(spec, y, LOSS_QUANTILE, np.array([1e-1, 1e-3]), foldid, 4, taus=taus, rounds=4, tol=1e-12,
                     maxit=400000)
    P, D, gap = o.duality_gap(spec, res, y, LOSS_QUANTILE)
    assert np.all(gap >= -1e-10) and np.all(gap <= 2 * res.smooth_final)
    rng = np.random.default_rng(1)
    for c in (0, 7, res.cols["B"] - 1):                    # weak duality against perturbed primal points
        M, lam, tau = res.cols["M"][:, c], res.cols["lam"][c], float(res.cols["tau"][c])
        alpha_c, b_c = o.path_coef(spec, res, c)
        for scale in (1e-2, 1.0):
            alpha = alpha_c + scale * rng.standard_normal(n) * np.abs(alpha_c).max()
            assert o.objective(K, y, alpha, b_c + scale, lam, LOSS_QUANTILE, mask=M, tau=tau, nominal=True) >= D[c] - 1e-10
    with pytest.raises(ValueError):
        o.duality_gap(spec, res, y, o.LOSS_LOGISTIC)
