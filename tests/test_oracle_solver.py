"""Pins P3-P6, P10-P12 for the oracle's solver.

Each test fixes the oracle against something other than itself: a dense linear solve, a
textbook linear system, the MM descent property, first-order optimality evaluated directly
from K (never through U), closed-form limits, or an independent Newton solve.
"""
import numpy as np
import pytest

import oracle as o
import workloads as wl
from oracle import LOSS_HINGE, LOSS_LOGISTIC, LOSS_QUANTILE, LOSS_DWD


def _problem(loss, n=50, p=4, seed=5):
    rng = np.random.default_rng(seed)
    if loss == LOSS_QUANTILE:
        X = rng.uniform(-1, 1, (n, p))
        y = np.sin(np.pi * X.sum(1) / np.sqrt(p)) + 0.3 * rng.standard_t(3, n)
    else:
        w = wl.config0(n=n, p=p, seed=seed)
        X, y = w.X, w.y
    sigma = wl.median_distance(X)
    K = o.gram_rbf(X, sigma)
    return X, y, K, o.spectral_setup(K), o.make_folds(n, 4, 3)


# ---------------------------------------------------------------- losses
def test_smoothed_hinge_matches_printed_formula():
    d = 0.25
    u = np.array([-2.0, 0.75, 0.9, 1.0, 1.2, 1.25, 3.0])
    want = np.array([3.0, 0.25, (0.9 - 1.25) ** 2, (1.0 - 1.25) ** 2, (1.2 - 1.25) ** 2, 0.0, 0.0])
    want[2:5] /= 4 * d
    got = o.smooth_loss(LOSS_HINGE, np.ones_like(u), u, d)
    assert np.allclose(got, want, atol=1e-15)
    # delta -> 0 recovers the hinge of eq. (1); L_delta - hinge in [0, delta/4]
    gap = got - np.maximum(1 - u, 0)
    assert np.all(gap >= -1e-15) and np.all(gap <= d / 4 + 1e-15)


@pytest.mark.parametrize("loss,smooth,tau", [(LOSS_HINGE, 0.3, None), (LOSS_LOGISTIC, None, None),
                                             (LOSS_QUANTILE, 0.2, 0.1), (LOSS_QUANTILE, 0.2, 0.9),
                                             (LOSS_DWD, None, None)])
def test_psi_is_derivative_and_curvature_bounds_it(loss, smooth, tau):
    rng = np.random.default_rng(1)
    y = np.where(rng.random(400) < 0.5, 1.0, -1.0) if loss != LOSS_QUANTILE else rng.standard_normal(400)
    f = 2.5 * rng.standard_normal(400)
    h = 1e-6
    num = (o.smooth_loss(loss, y, f + h, smooth, tau) - o.smooth_loss(loss, y, f - h, smooth, tau)) / (2 * h)
    assert np.max(np.abs(num - o.psi(loss, y, f, smooth, tau))) < 1e-5 / (smooth or 1.0)
    # second difference of the loss never exceeds the curvature constant (majoriser validity)
    f2 = np.linspace(-4, 4, 4001)
    yy = np.ones_like(f2) if loss != LOSS_QUANTILE else np.zeros_like(f2)
    p = o.psi(loss, yy, f2, smooth, tau)
    assert np.max(np.diff(p) / np.diff(f2)) <= o.curvature(loss, smooth) * (1 + 1e-9)
    assert np.min(np.diff(p)) >= -1e-15                                  # convex


def test_quantile_nominal_is_check_loss():
    t = np.array([-2.0, -0.5, 0.0, 0.5, 2.0])
    assert np.allclose(o.nominal_loss(LOSS_QUANTILE, t, 0 * t, 0.1), [1.8, 0.45, 0.0, 0.05, 0.2])
    # smoothed check loss is C^1 at +-gamma and within gamma/4 of the check loss
    g, tau = 0.3, 0.7
    tt = np.linspace(-1, 1, 2001)
    gap = o.smooth_loss(LOSS_QUANTILE, tt, 0 * tt, g, tau) - o.nominal_loss(LOSS_QUANTILE, tt, 0 * tt, tau)
    assert gap.min() >= -1e-15 and gap.max() <= g / 4 + 1e-15


# ---------------------------------------------------------------- P3: spectral step == dense solve
@pytest.mark.parametrize("loss,smooth,tau", [(LOSS_HINGE, 0.125, None), (LOSS_LOGISTIC, None, None),
                                             (LOSS_QUANTILE, 0.125, 0.3), (LOSS_DWD, None, None)])
def test_spectral_step_equals_dense_majoriser_solve(loss, smooth, tau):
    X, y, K, spec, foldid = _problem(loss, n=40)
    n = len(y)
    rng = np.random.default_rng(2)
    lam = 3e-3
    mask = (foldid != 1).astype(float)
    n_c = mask.sum()
    alpha_bar = 0.1 * rng.standard_normal(n)
    bbar = 0.2
    a_bar = spec.U.T @ alpha_bar
    c, S, s = o.column_constants(spec, lam, n_c, o.curvature(loss, smooth))
    # oracle step (as in fit_column)
    f = spec.U @ (spec.lam * a_bar) + bbar
    z = mask * o.psi(loss, y, f, smooth, tau) / n_c
    rho = spec.U.T @ z + 2 * lam * a_bar
    dbeta = (z.sum() - c * np.sum(S * spec.lam * spec.u1 * rho)) / s
    da = S * (rho - dbeta * c * spec.u1)
    # dense: P (dbeta; dalpha) = (1^T z ; K z + 2 lam K alpha)   (G1/G2)
    P = o.dense_majoriser(K, lam, c)
    fd = K @ alpha_bar + bbar
    zd = mask * o.psi(loss, y, fd, smooth, tau) / n_c
    rhs = np.concatenate([[zd.sum()], K @ zd + 2 * lam * K @ alpha_bar])
    got = np.concatenate([[dbeta], spec.U @ da])
    assert np.max(np.abs(P @ got - rhs)) < 1e-11 * max(1.0, np.abs(rhs).max())
    # and the paper's g as printed (no minus sign) does NOT satisfy it: G1
    g_printed = 1.0 / (n * np.sum(spec.u1 ** 2 * spec.lam ** 2 / (2 * lam * spec.lam + c * spec.lam ** 2 + 1e-300)))
    assert abs(g_printed - 1.0 / s) > 1e-3 * abs(1.0 / s)


# ---------------------------------------------------------------- P4: one step == LS-SVM system
def test_huge_delta_one_step_is_lssvm():
    X, y, K, spec, _ = _problem(LOSS_HINGE, n=45)
    n = len(y)
    lam, delta = 2e-2, 100.0
    a, b0, it, kkt, flag = o.fit_column(spec, y, LOSS_HINGE, [delta], lam, np.ones(n), maxit=1, momentum=False)
    A = np.zeros((n + 1, n + 1))
    A[0, 1:] = 1.0
    A[1:, 0] = 1.0
    A[1:, 1:] = K + 4 * delta * n * lam * np.eye(n)
    sol = np.linalg.solve(A, np.concatenate([[0.0], (1 + delta) * y]))
    assert abs(b0 - sol[0]) < 1e-9 * max(1, abs(sol[0]))
    assert np.max(np.abs(spec.U @ a - sol[1:])) < 1e-9 * np.abs(sol[1:]).max()


def test_huge_gamma_one_step_is_least_squares_kqr():
    X, y, K, spec, _ = _problem(LOSS_QUANTILE, n=45)
    n = len(y)
    lam, gam, tau = 1e-2, 100.0, 0.3
    a, b0, *_ = o.fit_column(spec, y, LOSS_QUANTILE, [gam], lam, np.ones(n), tau=tau, maxit=1, momentum=False)
    A = np.zeros((n + 1, n + 1))
    A[0, 1:] = 1.0
    A[1:, 0] = 1.0
    A[1:, 1:] = K + 4 * gam * n * lam * np.eye(n)
    sol = np.linalg.solve(A, np.concatenate([[0.0], y + 2 * gam * (tau - 0.5)]))
    assert abs(b0 - sol[0]) < 1e-9 * max(1, abs(sol[0]))
    assert np.max(np.abs(spec.U @ a - sol[1:])) < 1e-9 * np.abs(sol[1:]).max()


# ---------------------------------------------------------------- P5: MM descent
@pytest.mark.parametrize("loss,smooth,tau", [(LOSS_HINGE, 0.125, None), (LOSS_LOGISTIC, None, None),
                                             (LOSS_QUANTILE, 0.125, 0.9), (LOSS_DWD, None, None)])
def test_objective_never_increases_without_momentum(loss, smooth, tau):
    X, y, K, spec, foldid = _problem(loss, n=40)
    mask = (foldid != 0).astype(float)
    lam = 1e-3
    trace = []
    o.fit_column(spec, y, loss, [smooth], lam, mask, tau=tau, maxit=60, momentum=False, trace=trace)
    vals = [o.objective(K, y, spec.U @ ab, bb, lam, loss, mask, smooth, tau) for (_, _, ab, bb) in trace]
    assert len(vals) == 60
    assert np.all(np.diff(vals) <= 1e-13 * max(1.0, abs(vals[0])))
    assert vals[-1] < vals[0]


# ---------------------------------------------------------------- P6: KKT at convergence
@pytest.mark.parametrize("loss,taus", [(LOSS_HINGE, ()), (LOSS_LOGISTIC, ()), (LOSS_QUANTILE, (0.1, 0.5, 0.9)),
                                       (LOSS_DWD, ())])
def test_kkt_of_every_path_solution(loss, taus):
    X, y, K, spec, foldid = _problem(loss, n=48)
    lambdas = wl.lambda_grid(0, -4, 4)
    V = 4
    res = o.fit_path(spec, y, loss, lambdas, foldid, V, taus=taus, smooth0=1.0, eta=0.125, rounds=3,
                     tol=1e-12, maxit=100000)
    assert res.flags.sum() == 0
    cols = res.cols
    for c in range(cols["B"]):
        lam, M, n_c = cols["lam"][c], cols["M"][:, c], cols["n_c"][c]
        tau = cols["tau"][c] if loss == LOSS_QUANTILE else None
        alpha = spec.U @ res.a[:, c]
        f = K @ alpha + res.beta0[c]                                   # straight from K, not U
        z = M * o.psi(loss, y, f, res.smooth_final, tau) / n_c
        assert abs(z.sum()) < 1e-11                                    # d/d beta0 = 1^T z = 0
        assert np.max(np.abs(z + 2 * lam * alpha)) * n_c < 1e-9        # alpha = -z / (2 lam)
        assert abs(alpha.sum()) * 2 * lam * n_c < 1e-9                 # sum alpha = 0
        w2 = 2 * lam * n_c * alpha
        if loss == LOSS_QUANTILE:
            assert np.all(w2 >= tau - 1 - 1e-9) and np.all(w2 <= tau + 1e-9)
        else:
            assert np.all(y * w2 >= -1e-9) and np.all(y * w2 <= 1 + 1e-9)
        assert np.all(np.abs(alpha[M == 0]) * 2 * lam * n_c < 1e-9)    # P8: held-out alpha = 0


@pytest.mark.parametrize("loss,taus", [(LOSS_HINGE, ()), (LOSS_LOGISTIC, ()), (LOSS_QUANTILE, (0.3, 0.8))])
def test_column_mode_and_batched_mode_agree_on_every_column(loss, taus):
    """fit_path (the mode the GPU parity tests call) against fit_column (Algorithm 1 column by column, mat-vecs):
    every column of a small grid, both at tol = 1e-13, to the 1e-10 coefficient bar the parity tests use."""
    X, y, K, spec, foldid = _problem(loss, n=48)
    lambdas = wl.lambda_grid(0, -3, 4)
    V = 4
    res = o.fit_path(spec, y, loss, lambdas, foldid, V, taus=taus, smooth0=1.0, eta=0.125, rounds=3,
                     tol=1e-13, maxit=400000)
    assert res.flags.sum() == 0
    cols = res.cols
    levels = o.smoothing_levels(loss, 1.0, 0.125, 3)
    for c in range(cols["B"]):
        tau = cols["tau"][c] if loss == LOSS_QUANTILE else None
        a, b0, it, kkt, flag = o.fit_column(spec, y, loss, levels, cols["lam"][c], cols["M"][:, c], tau=tau,
                                            tol=1e-13, maxit=400000)
        assert flag == 0
        al, al2 = spec.U @ a, spec.U @ res.a[:, c]
        assert np.linalg.norm(al - al2) <= 1e-10 * np.linalg.norm(al2), c
        assert abs(b0 - res.beta0[c]) <= 1e-10 * max(1.0, abs(b0)), c
        assert abs(it - res.iters[c]) <= max(3, 0.05 * it)     # same arithmetic up to the summation order of BLAS


def test_logistic_against_independent_newton():
    """Independent solve of the stationarity equations alpha + z(K alpha + b)/(2 lam) = 0,
    1^T z = 0 by Newton's method on the dense system (no eigendecomposition, no MM)."""
    X, y, K, spec, foldid = _problem(LOSS_LOGISTIC, n=40)
    n = len(y)
    lam = 5e-3
    mask = (foldid != 2).astype(float)
    n_c = mask.sum()
    a, b0, *_ = o.fit_column(spec, y, LOSS_LOGISTIC, [None], lam, mask, tol=1e-13, maxit=100000)
    alpha, beta = np.zeros(n), 0.0
    for _ in range(50):
        f = K @ alpha + beta
        sg = 1.0 / (1.0 + np.exp(y * f))
        z = mask * (-y * sg) / n_c
        D = mask * sg * (1 - sg) / n_c                                 # d z / d f
        G = np.concatenate([alpha + z / (2 * lam), [z.sum()]])
        J = np.zeros((n + 1, n + 1))
        J[:n, :n] = np.eye(n) + (D[:, None] * K) / (2 * lam)
        J[:n, n] = D / (2 * lam)
        J[n, :n] = D @ K
        J[n, n] = D.sum()
        step = np.linalg.solve(J, G)
        alpha -= step[:n]
        beta -= step[n]
        if np.max(np.abs(step)) < 1e-14:
            break
    assert np.linalg.norm(spec.U @ a - alpha) < 1e-9 * np.linalg.norm(alpha)
    assert abs(b0 - beta) < 1e-9


def test_hinge_against_scipy_minimiser():
    """Objective value of the converged smoothed-hinge fit vs a generic quasi-Newton
    minimiser of the same objective in (beta0, a) coordinates."""
    from scipy.optimize import minimize
    X, y, K, spec, foldid = _problem(LOSS_HINGE, n=30)
    n = len(y)
    lam, delta = 1e-2, 0.125
    mask = (foldid != 0).astype(float)
    a, b0, *_ = o.fit_column(spec, y, LOSS_HINGE, [delta], lam, mask, tol=1e-12, maxit=100000)
    mine = o.objective(K, y, spec.U @ a, b0, lam, LOSS_HINGE, mask, delta)

    def fun(x):
        return o.objective(K, y, x[1:], x[0], lam, LOSS_HINGE, mask, delta)
    best = minimize(fun, np.zeros(n + 1), method="BFGS", options=dict(gtol=1e-10, maxiter=5000))
    assert mine <= best.fun + 1e-12
    assert best.fun - mine < 1e-7


# ---------------------------------------------------------------- P10: large-lambda limit
def test_large_lambda_limit_closed_forms():
    n = 60
    rng = np.random.default_rng(8)
    X = rng.standard_normal((n, 3))
    K = o.gram_rbf(X, 1.5)
    spec = o.spectral_setup(K)
    y = np.ones(n)
    y[:21] = -1.0                                                      # n+ = 39, n- = 21
    lam = 1e7
    ones = np.ones(n)
    delta = 0.125
    a, b0, *_ = o.fit_column(spec, y, LOSS_HINGE, [delta], lam, ones, tol=1e-13, maxit=100000)
    assert b0 == pytest.approx(1 + delta - 2 * delta * 21 / 39, abs=1e-5)
    alpha = spec.U @ a
    assert np.max(np.abs(alpha)) < 1e-6
    assert np.allclose(2 * lam * n * alpha, -o.psi(LOSS_HINGE, y, b0 * ones, delta), atol=1e-4)
    a, b0, *_ = o.fit_column(spec, y, LOSS_LOGISTIC, [None], lam, ones, tol=1e-13, maxit=100000)
    assert b0 == pytest.approx(np.log(39 / 21), abs=1e-5)
    yq = rng.standard_normal(n)
    g, tau = 0.05, 0.3
    a, b0, *_ = o.fit_column(spec, yq, LOSS_QUANTILE, [g], lam, ones, tau=tau, tol=1e-13, maxit=100000)
    # root of sum_j H'(y_j - b0) = 0
    t = yq - b0
    hp = np.where(t < -g, tau - 1, np.where(t > g, tau, t / (2 * g) + tau - 0.5))
    assert abs(hp.sum()) < 1e-4
    assert abs(np.mean(t < 0) - tau) <= (np.sum(np.abs(t) <= g) + 1) / n      # P11


# ---------------------------------------------------------------- P11, P12
def test_kqr_residual_fraction_and_path_ordering():
    X, y, K, spec, foldid = _problem(LOSS_QUANTILE, n=80, seed=9)
    n = len(y)
    lambdas = wl.lambda_grid(-1, -4, 5)
    taus = (0.1, 0.5, 0.9)
    res = o.fit_path(spec, y, LOSS_QUANTILE, lambdas, foldid, 4, taus=taus, rounds=4, tol=1e-11, maxit=200000)
    cols = res.cols
    g = res.smooth_final
    for t, tau in enumerate(taus):
        pen, fit = [], []
        for l in range(5):
            c = (t * 5 + 4) * 5 + l                                    # v = V: no fold held out
            alpha = spec.U @ res.a[:, c]
            f = K @ alpha + res.beta0[c]
            r = y - f
            assert abs(np.mean(r < 0) - tau) <= (np.sum(np.abs(r) <= g) + 1) / n   # P11
            pen.append(alpha @ K @ alpha)
            fit.append(np.mean(o.smooth_loss(LOSS_QUANTILE, y, f, g, tau)))
        # lambdas descending: penalty non-decreasing, training loss non-increasing (P12)
        assert np.all(np.diff(pen) >= -1e-9) and np.all(np.diff(fit) <= 1e-9)


# ---------------------------------------------------------------- DWD (reading G20)
def test_dwd_loss_matches_its_definition_and_limits():
    """Generalised DWD loss with q = 1 (Wang and Zou 2018, cited at PAPER.md:81): linear for u <= 1/2, 1/(4u)
    beyond; C^1 at the joint, convex, and the large-lambda intercept has a closed form."""
    u = np.array([-2.0, 0.0, 0.5, 0.5 + 1e-9, 1.0, 4.0])
    got = o.smooth_loss(LOSS_DWD, np.ones_like(u), u)
    assert np.allclose(got, [3.0, 1.0, 0.5, 0.5, 0.25, 0.0625], atol=1e-8)
    assert np.allclose(o.psi(LOSS_DWD, np.ones(3), np.array([0.5 - 1e-12, 0.5 + 1e-12, 1.0])), [-1.0, -1.0, -0.25])
    grid = np.linspace(0.5, 6.0, 4001)
    curv = np.diff(o.psi(LOSS_DWD, np.ones_like(grid), grid)) / np.diff(grid)
    assert curv.max() <= o.curvature(LOSS_DWD, None) + 1e-6 and curv.max() > 3.9 and curv.min() >= 0
    # large lambda: alpha -> 0 and beta0 solves n+ V'(b) = n- V'(-b); for n+ > n-: b = sqrt(n+/n-)/2 > 1/2
    n = 60
    rng = np.random.default_rng(8)
    K = o.gram_rbf(rng.standard_normal((n, 3)), 1.5)
    spec = o.spectral_setup(K)
    y = np.ones(n)
    y[:21] = -1.0
    a, b0, *_ = o.fit_column(spec, y, LOSS_DWD, [None], 1e7, np.ones(n), tol=1e-13, maxit=100000)
    assert abs(b0 - 0.5 * np.sqrt(39.0 / 21.0)) < 1e-6
    assert np.abs(spec.U @ a).max() < 1e-6


def test_dwd_against_scipy_minimiser():
    from scipy.optimize import minimize
    X, y, K, spec, foldid = _problem(LOSS_DWD, n=30)
    n = len(y)
    lam = 1e-2
    mask = (foldid != 0).astype(float)
    a, b0, *_ = o.fit_column(spec, y, LOSS_DWD, [None], lam, mask, tol=1e-12, maxit=100000)
    mine = o.objective(K, y, spec.U @ a, b0, lam, LOSS_DWD, mask, None)
    best = minimize(lambda x: o.objective(K, y, x[1:], x[0], lam, LOSS_DWD, mask, None), np.zeros(n + 1),
                    method="BFGS", options=dict(gtol=1e-10, maxiter=5000))
    assert mine <= best.fun + 1e-12 and best.fun - mine < 1e-7


# ---------------------------------------------------------------- warm-start rounds (an input, not a result)
def test_warm_tol_does_not_move_the_result():
    """Rounds 0..R-2 only produce starting points: a loose warm_tol changes the iteration counts, not the
    minimiser at the final level (both stopped at the same tol)."""
    X, y, K, spec, foldid = _problem(LOSS_HINGE, n=60)
    lambdas = wl.lambda_grid(0, -3, 4)
    r0 = o.fit_path(spec, y, LOSS_HINGE, lambdas, foldid, 4, rounds=4, tol=1e-13, maxit=400000)
    r1 = o.fit_path(spec, y, LOSS_HINGE, lambdas, foldid, 4, rounds=4, tol=1e-13, maxit=400000, warm_tol=1e-3)
    assert r0.flags.sum() == 0 and r1.flags.sum() == 0
    assert r1.iters.sum() < r0.iters.sum()
    for c in range(r0.cols["B"]):
        a0, a1 = spec.U @ r0.a[:, c], spec.U @ r1.a[:, c]
        assert np.linalg.norm(a0 - a1) <= 1e-10 * np.linalg.norm(a0)


# ---------------------------------------------------------------- P18: outer control (reading G23)
def test_outer_control_gap_tol_zero_is_the_fixed_schedule():
    X, y, K, spec, foldid = _problem(LOSS_HINGE, n=48)
    lambdas = wl.lambda_grid(0, -3, 3)
    r0 = o.fit_path(spec, y, LOSS_HINGE, lambdas, foldid, 4, rounds=3, tol=1e-12, maxit=200000)
    r1 = o.fit_path(spec, y, LOSS_HINGE, lambdas, foldid, 4, rounds=3, tol=1e-12, maxit=200000, gap_tol=0.0)
    assert np.array_equal(r0.a, r1.a) and np.array_equal(r0.beta0, r1.beta0) and np.all(r1.level == 2)


@pytest.mark.parametrize("loss,taus,warm_tol", [(LOSS_HINGE, (), None), (LOSS_HINGE, (), 1e-3),
                                                (LOSS_QUANTILE, (0.2, 0.7), 1e-3)])
def test_outer_control_exits_at_the_first_level_that_certifies_the_gap(loss, taus, warm_tol):
    """Every column ends on the FIRST level k whose warm-started iterate certifies gap <= gap_tol (or on the
    cap R-1), its coefficients are the minimiser at that level (== the fixed schedule with k+1 rounds), and the
    certificate holds for the returned solution."""
    X, y, K, spec, foldid = _problem(loss, n=56)
    lambdas = wl.lambda_grid(0, -3, 4)
    V, R, gap_tol = 4, 4, 3e-3
    res = o.fit_path(spec, y, loss, lambdas, foldid, V, taus=taus, rounds=R, tol=1e-12, maxit=400000,
                     warm_tol=warm_tol, gap_tol=gap_tol)
    assert res.flags.sum() == 0
    assert len(set(res.level.tolist())) >= 2, "choose gap_tol so that the test sees several exit levels"
    fixed = {k: o.fit_path(spec, y, loss, lambdas, foldid, V, taus=taus, rounds=k + 1, tol=1e-12, maxit=400000)
             for k in range(R)}
    gaps = {k: o.duality_gap(spec, fixed[k], y, loss)[2] for k in range(R)}
    P, D, gap = o.duality_gap(spec, res, y, loss)
    for c in range(res.cols["B"]):
        k = int(res.level[c])
        ref = fixed[k]
        a0, a1 = spec.U @ ref.a[:, c], spec.U @ res.a[:, c]
        assert np.linalg.norm(a0 - a1) <= 1e-9 * max(np.linalg.norm(a0), 1e-300), (c, k)
        assert abs(gap[c] - gaps[k][c]) <= 1e-9
        if k < R - 1:
            assert gap[c] <= gap_tol + 1e-9
        # no earlier level's minimiser carries the certificate; with warm_tol the screen runs on an iterate that is
        # only within warm_tol of that minimiser, so a near miss may stay on the schedule (conservative, still valid)
        for j in range(k):
            assert gaps[j][c] > gap_tol * (1.0 if warm_tol is None else 0.7), (c, j)
    # column mode takes the same decisions
    levels = o.smoothing_levels(loss, 1.0, 0.125, R)
    for c in (0, res.cols["B"] // 3, res.cols["B"] - 1):
        tau = res.cols["tau"][c] if loss == LOSS_QUANTILE else None
        a, b0, it, kkt, flag, lev = o.fit_column(spec, y, loss, levels, res.cols["lam"][c], res.cols["M"][:, c],
                                                 tau=tau, tol=1e-12, maxit=400000, warm_tol=warm_tol,
                                                 gap_tol=gap_tol, want_level=True)
        assert lev == res.level[c] and abs(it - res.iters[c]) <= max(3, 0.05 * it)
        assert np.linalg.norm(a - res.a[:, c]) <= 1e-10 * max(np.linalg.norm(a), 1e-300)


def test_outer_control_certificate_against_svc():
    """The exit test certifies the ORIGINAL problem: P(returned alpha) - P*(scikit-learn SVC dual solver) <= gap_tol
    for every column that left the schedule early (C = 1/(2 n lambda))."""
    from sklearn.svm import SVC
    n = 72
    X, y, K, spec, _ = _problem(LOSS_HINGE, n=n)
    foldid = np.zeros(n, dtype=np.int64)
    foldid[::2] = 1
    lambdas = np.array([3e-2, 3e-3])
    gap_tol = 5e-3
    res = o.fit_path(spec, y, LOSS_HINGE, lambdas, foldid, 2, rounds=5, tol=1e-12, maxit=400000, warm_tol=1e-3,
                     gap_tol=gap_tol)
    early = 0
    for l, lam in enumerate(lambdas):
        c = 2 * len(lambdas) + l                          # v = V: the full-data column
        svc = SVC(C=1.0 / (2 * n * lam), kernel="precomputed", tol=1e-10).fit(K, y)
        alpha_qp = np.zeros(n)
        alpha_qp[svc.support_] = svc.dual_coef_[0]
        p_star = o.objective(K, y, alpha_qp, float(svc.intercept_[0]), lam, LOSS_HINGE, nominal=True)
        alpha, b0 = o.path_coef(spec, res, c)
        p = o.objective(K, y, alpha, b0, lam, LOSS_HINGE, nominal=True)
        assert p >= p_star - 1e-8
        if res.level[c] < 4:
            early += 1
            assert p - p_star <= gap_tol + 1e-8
    assert early >= 1


def test_outer_control_huge_gap_tol_stops_after_the_first_round():
    X, y, K, spec, foldid = _problem(LOSS_HINGE, n=40)
    lambdas = wl.lambda_grid(0, -2, 3)
    res = o.fit_path(spec, y, LOSS_HINGE, lambdas, foldid, 4, rounds=4, tol=1e-12, maxit=200000, gap_tol=10.0)
    one = o.fit_path(spec, y, LOSS_HINGE, lambdas, foldid, 4, rounds=1, tol=1e-12, maxit=200000)
    assert np.all(res.level == 0) and np.array_equal(res.a, one.a)


# ---------------------------------------------------------------- warm starts along lambda, measured
def test_lambda_warm_start_against_delta_warm_start():
    """DESIGN.md section 8 keeps warm starts along delta and batches all lambda at once.  Measured here on the
    oracle: the last smoothing round started from the converged NEIGHBOUR-lambda solution (the paper's
    lambda-sequential order) needs at least as many iterations, summed over the small-lambda half of
    the grid, as started from the same column's previous smoothing round."""
    w = wl.config0(n=300, p=10, L=12, seed=1000)
    K = o.gram_rbf(w.X, float(w.sigmas[0]))
    spec = o.spectral_setup(K)
    mask = np.ones(w.n)
    levels = o.smoothing_levels(LOSS_HINGE, 1.0, 0.125, 4)
    it_delta, it_lambda = [], []
    prev = None
    for l, lam in enumerate(w.lambdas):
        aw, bw, *_ = o.fit_column(spec, w.y, LOSS_HINGE, levels[:-1], lam, mask, tol=1e-3, maxit=100000)
        a, b, it, *_ = o.fit_column(spec, w.y, LOSS_HINGE, levels[-1:], lam, mask, tol=1e-10, maxit=200000, a0=aw, b0=bw)
        it_delta.append(it)
        if prev is not None:
            _, _, it2, *_ = o.fit_column(spec, w.y, LOSS_HINGE, levels[-1:], lam, mask, tol=1e-10, maxit=200000,
                                         a0=prev[0], b0=prev[1])
            it_lambda.append(it2)
        prev = (a, b)
    half = len(w.lambdas) // 2
    print("iterations of the last round, delta warm start: %s; lambda warm start: %s" % (it_delta[1:], it_lambda))
    assert sum(it_lambda[half - 1:]) >= 0.9 * sum(it_delta[half:])
