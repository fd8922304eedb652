"""Pins of the Platt-scaling oracle (reading G21): first-order optimality of the fitted sigmoid, agreement with
scikit-learn's independent implementation of the same method, and the held-out decision values it is fed."""
import numpy as np

import oracle as o
import workloads as wl


def _scores(n=400, seed=3):
    rng = np.random.default_rng(seed)
    y = np.where(rng.random(n) < 0.4, 1.0, -1.0)
    f = 1.3 * y + rng.standard_normal(n) + 0.2
    return f, y


def test_platt_gradient_vanishes_at_solution():
    f, y = _scores()
    A, B = o.platt_fit(f, y)
    t, *_ = o.platt_targets(y)
    p = o.platt_proba(f, A, B)
    assert abs(np.sum(f * (t - p))) < 1e-5 and abs(np.sum(t - p)) < 1e-5
    assert A < 0                                     # larger score -> larger P(y = +1)
    h = 1e-5                                         # and it is a minimum of the printed objective
    base = o.platt_objective(f, t, A, B)
    for dA, dB in ((h, 0), (-h, 0), (0, h), (0, -h)):
        assert o.platt_objective(f, t, A + dA, B + dB) >= base - 1e-12


def test_platt_matches_sklearn_sigmoid_calibration():
    from sklearn.calibration import _sigmoid_calibration
    for seed in (1, 2):
        f, y = _scores(seed=seed)
        A, B = o.platt_fit(f, y)
        As, Bs = _sigmoid_calibration(f, (y > 0).astype(float))
        p, ps = o.platt_proba(f, A, B), 1.0 / (1.0 + np.exp(As * f + Bs))
        assert np.max(np.abs(p - ps)) < 1e-4


def test_platt_is_equivariant_under_affine_scores():
    f, y = _scores(seed=5)
    A, B = o.platt_fit(f, y)
    A2, B2 = o.platt_fit(3.0 * f - 1.0, y)
    assert np.max(np.abs(o.platt_proba(f, A, B) - o.platt_proba(3.0 * f - 1.0, A2, B2))) < 1e-5


def test_cv_decision_values_are_the_refit_predictions():
    w = wl.config0(n=60, p=4, L=3, V=3, seed=9)
    sigma = float(w.sigmas[0])
    foldid = o.make_folds(w.n, w.V, w.fold_seed)
    K = o.gram_rbf(w.X, sigma)
    spec = o.spectral_setup(K)
    res = o.fit_path(spec, w.y, w.loss, w.lambdas, foldid, w.V, rounds=2, tol=1e-12, maxit=200000)
    l = 1
    f = o.cv_decision_values(spec, res, foldid, 0, l, w.L, w.V)
    for v in range(w.V):
        act, alpha_act, b0, f_out, rows = o.brute_force_refit(K, w.y, foldid, v, w.lambdas[l], w.loss,
                                                              o.smoothing_levels(w.loss, 1.0, 0.125, 2),
                                                              tol=1e-12, maxit=200000)
        assert np.max(np.abs(f_out - f[rows])) < 1e-8
