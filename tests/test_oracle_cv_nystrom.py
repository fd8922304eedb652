"""Pins P7-P9, P13, P15 for the oracle: exact CV == brute-force refit, the hinge limit
against an independent QP solver, Nystrom special cases, prediction."""
import numpy as np
import pytest

import oracle as o
import workloads as wl
from oracle import LOSS_HINGE, LOSS_LOGISTIC, LOSS_QUANTILE, LOSS_DWD


def _data(loss, n, p=4, seed=21):
    rng = np.random.default_rng(seed)
    if loss == LOSS_QUANTILE:
        X = rng.uniform(-1, 1, (n, p))
        y = np.sin(np.pi * X.sum(1) / np.sqrt(p)) + 0.3 * rng.standard_t(3, n)
    else:
        w = wl.config0(n=n, p=p, seed=seed)
        X, y = w.X, w.y
    return X, y, wl.median_distance(X)


# ------------------------------------------------------------ P7 / P8
@pytest.mark.parametrize("loss,taus,rounds", [(LOSS_HINGE, (), 3), (LOSS_LOGISTIC, (), 1),
                                              (LOSS_QUANTILE, (0.1, 0.9), 3), (LOSS_DWD, (), 1)])
def test_exact_cv_equals_brute_force_refit(loss, taus, rounds):
    n, V = 64, 4
    X, y, sigma = _data(loss, n)
    K = o.gram_rbf(X, sigma)
    spec = o.spectral_setup(K)
    foldid = o.make_folds(n, V, 5)
    lambdas = np.array([1e-1, 1e-2, 1e-3])
    res = o.fit_path(spec, y, loss, lambdas, foldid, V, taus=taus, rounds=rounds, tol=1e-12, maxit=200000)
    assert res.flags.sum() == 0
    cv_loss, cv_err, cv_mean, best = o.exact_cv(spec, res, y, foldid, loss, taus)
    levels = o.smoothing_levels(loss, 1.0, 0.125, rounds)
    T = max(1, len(taus))
    for t in range(T):
        tau = taus[t] if taus else None
        for v in range(V):
            for l, lam in enumerate(lambdas):
                act, alpha_r, b_r, f_r, rows = o.brute_force_refit(K, y, foldid, v, lam, loss, levels, tau=tau)
                c = (t * (V + 1) + v) * len(lambdas) + l
                alpha_full = spec.U @ res.a[:, c]
                scale = max(1.0, np.abs(alpha_r).max())
                assert np.max(np.abs(alpha_full[act] - alpha_r)) < 2e-8 * scale     # same training coefficients
                assert np.max(np.abs(alpha_full[rows])) < 2e-8 * scale              # P8: held-out alpha -> 0
                if loss == LOSS_HINGE:
                    # G18: beta0 is not unique when every training row sits on the linear piece
                    # of L_delta and the training labels are balanced; compare what is unique.
                    u = y[act] * (K[np.ix_(act, act)] @ alpha_r + b_r)
                    if np.all(u <= 1 - levels[-1]) and y[act].sum() == 0:
                        Ka = K[np.ix_(act, act)]
                        o1 = o.objective(Ka, y[act], alpha_r, b_r, lam, loss, None, levels[-1])
                        o2 = o.objective(Ka, y[act], alpha_full[act], res.beta0[c], lam, loss, None, levels[-1])
                        assert abs(o1 - o2) < 1e-12
                        continue
                assert abs(res.beta0[c] - b_r) < 2e-8
                f_masked = K[rows] @ alpha_full + res.beta0[c]
                assert np.max(np.abs(f_masked - f_r)) < 1e-7
                want = np.mean(o.nominal_loss(loss, y[rows], f_r, tau))
                assert abs(cv_loss[t, l, v] - want) < 1e-7
                if loss != LOSS_QUANTILE:
                    assert cv_err[t, l, v] == int(np.sum(o.label_of(f_r) != y[rows]))
    # pooled mean and argmin with the tie rule (G14)
    sizes = np.bincount(foldid, minlength=V)
    assert np.allclose(cv_mean, (cv_loss * sizes).sum(2) / n)
    for t in range(T):
        assert best[t] == int(np.argmin(cv_mean[t]))


def test_cv_tie_break_prefers_largest_lambda():
    # two lambdas so large that both fits are the constant model: identical CV losses
    n, V = 40, 4
    X, y, sigma = _data(LOSS_LOGISTIC, n, seed=4)
    spec = o.spectral_setup(o.gram_rbf(X, sigma))
    foldid = o.make_folds(n, V, 1)
    lambdas = np.array([1e9, 1e8])
    res = o.fit_path(spec, y, LOSS_LOGISTIC, lambdas, foldid, V, rounds=1, tol=1e-13, maxit=100000)
    res.a[:] = 0.0                        # exact constant models => exactly tied scores
    res.beta0[: len(res.beta0)] = np.repeat(res.beta0.reshape(V + 1, 2)[:, :1], 2, axis=1).ravel()
    *_, cv_mean, best = o.exact_cv(spec, res, y, foldid, LOSS_LOGISTIC)
    assert cv_mean[0, 0] == cv_mean[0, 1] and best[0] == 0


# ------------------------------------------------------------ P9 / P15
def test_hinge_limit_against_sklearn_svc():
    from sklearn.svm import SVC
    n = 80
    X, y, sigma = _data(LOSS_HINGE, n, seed=33)
    K = o.gram_rbf(X, sigma)
    spec = o.spectral_setup(K)
    ones = np.ones(n)
    for lam in (1e-2, 1e-3):
        C = 1.0 / (2 * n * lam)
        svc = SVC(C=C, kernel="precomputed", tol=1e-10).fit(K, y)
        alpha_qp = np.zeros(n)
        alpha_qp[svc.support_] = svc.dual_coef_[0]
        f_qp = svc.decision_function(K)
        obj_qp = o.objective(K, y, alpha_qp, float(svc.intercept_[0]), lam, LOSS_HINGE, nominal=True)
        # P15: C sum hinge + 1/2 a^T K a == (1/(2 lam)) [(1/n) sum hinge + lam a^T K a]
        sk_obj = C * np.sum(np.maximum(1 - y * f_qp, 0)) + 0.5 * alpha_qp @ K @ alpha_qp
        assert sk_obj == pytest.approx(obj_qp / (2 * lam), rel=1e-10)
        prev_gap, a, b0 = None, None, 0.0
        for k in range(5):
            delta = 0.125 ** k
            a, b0, *_ = o.fit_column(spec, y, LOSS_HINGE, [delta], lam, ones, tol=1e-11, maxit=400000, a0=a, b0=b0)
            alpha = spec.U @ a
            obj = o.objective(K, y, alpha, b0, lam, LOSS_HINGE, nominal=True)
            # L_delta - hinge in [0, delta/4]  =>  0 <= obj(x_delta) - obj(x_qp) <= delta/4
            assert -1e-7 <= obj - obj_qp <= delta / 4 + 1e-7
            gap = np.max(np.abs(K @ alpha + b0 - f_qp))
            if prev_gap is not None and prev_gap > 1e-5:
                assert gap < prev_gap
            prev_gap = gap
        assert prev_gap < 10 * 0.125 ** 4                               # max|f_delta - f_qp| <~ delta


# ------------------------------------------------------------ P13 (reading G11)
def test_nystrom_all_landmarks_equals_full_kernel():
    n, V = 50, 5
    X, y, sigma = _data(LOSS_HINGE, n, seed=2)
    K = o.gram_rbf(X, sigma)
    full = o.spectral_setup(K)
    nys = o.nystrom_setup(X, sigma, np.arange(n))
    assert np.max(np.abs((nys.U * nys.lam) @ nys.U.T - K)) < 1e-8
    foldid = o.make_folds(n, V, 9)
    lambdas = np.array([1e-1, 1e-2])
    r1 = o.fit_path(full, y, LOSS_HINGE, lambdas, foldid, V, rounds=2, tol=1e-12, maxit=200000)
    r2 = o.fit_path(nys, y, LOSS_HINGE, lambdas, foldid, V, rounds=2, tol=1e-12, maxit=200000)
    for c in range(r1.cols["B"]):
        f1 = full.U @ (full.lam * r1.a[:, c]) + r1.beta0[c]
        f2 = nys.U @ (nys.lam * r2.a[:, c]) + r2.beta0[c]
        assert np.max(np.abs(f1 - f2)) < 1e-6
    cv1 = o.exact_cv(full, r1, y, foldid, LOSS_HINGE)
    cv2 = o.exact_cv(nys, r2, y, foldid, LOSS_HINGE)
    assert np.max(np.abs(cv1[0] - cv2[0])) < 1e-6 and np.array_equal(cv1[3], cv2[3])


def test_nystrom_thin_u_equals_eigh_of_low_rank_kernel():
    n, m, V = 70, 12, 4
    X, y, sigma = _data(LOSS_LOGISTIC, n, seed=6)
    idx = wl.landmarks(n, m, 3)
    nys = o.nystrom_setup(X, sigma, idx)
    assert nys.r <= m and np.max(np.abs(nys.U.T @ nys.U - np.eye(nys.r))) < 1e-10
    # K~ = K_nm K_mm^+ K_mn, the textbook Nystrom approximation
    K_nm = o.gram_rbf(X, sigma, X[idx])
    Kt = K_nm @ np.linalg.pinv(o.gram_rbf(X[idx], sigma), rcond=1e-12, hermitian=True) @ K_nm.T
    assert np.max(np.abs((nys.U * nys.lam) @ nys.U.T - Kt)) < 1e-8
    dense = o.spectral_setup(Kt)                   # full n x n decomposition of the same K~
    foldid = o.make_folds(n, V, 2)
    lambdas = np.array([1e-2, 1e-3])
    r_thin = o.fit_path(nys, y, LOSS_LOGISTIC, lambdas, foldid, V, rounds=1, tol=1e-12, maxit=200000)
    r_full = o.fit_path(dense, y, LOSS_LOGISTIC, lambdas, foldid, V, rounds=1, tol=1e-12, maxit=200000)
    for c in range(r_thin.cols["B"]):
        f1 = nys.U @ (nys.lam * r_thin.a[:, c]) + r_thin.beta0[c]
        f2 = dense.U @ (dense.lam * r_full.a[:, c]) + r_full.beta0[c]
        assert np.max(np.abs(f1 - f2)) < 1e-7
    # landmark weights reproduce the training decision values and predict new points
    c = r_thin.cols["B"] - 1
    gam = o.nystrom_landmark_weights(nys, r_thin.a[:, c])
    f_train = nys.U @ (nys.lam * r_thin.a[:, c]) + r_thin.beta0[c]
    f_lm, lab = o.predict(X[idx], gam, r_thin.beta0[c], sigma, X)
    assert np.max(np.abs(f_lm - f_train)) < 1e-7 and np.array_equal(lab, o.label_of(f_train))


def test_predict_full_kernel_reproduces_training_values():
    n = 40
    X, y, sigma = _data(LOSS_HINGE, n, seed=12)
    K = o.gram_rbf(X, sigma)
    spec = o.spectral_setup(K)
    foldid = o.make_folds(n, 4, 2)
    res = o.fit_path(spec, y, LOSS_HINGE, np.array([1e-2]), foldid, 4, rounds=2, tol=1e-11, maxit=100000)
    alpha, b0 = o.path_coef(spec, res, res.cols["B"] - 1)
    f, lab = o.predict(X, alpha, b0, sigma, X)
    assert np.max(np.abs(f - (K @ alpha + b0))) < 1e-12
    assert lab.dtype == np.int8 and set(np.unique(lab)) <= {-1, 1}
    assert o.label_of(np.array([0.0, -0.0, -1e-300]))[0] == 1          # G15: label(0) = +1
