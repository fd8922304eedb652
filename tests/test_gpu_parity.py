"""GPU parity tests: the CUDA path (through the C ABI of libtkm.so) against the FP64 oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json's: coefficients relative l2 <= 1e-10
(FP64 path), CV loss per (lambda, fold) within 1e-5, selected lambda identical, fold assignments and
predicted labels bit-exact.  Where several results are correct (U; beta0 of a degenerate column,
reading G18) only what is unique is compared."""
import numpy as np
import pytest

import oracle as o
import workloads as wl

pytestmark = pytest.mark.gpu

COEF_TOL_F64 = 1e-10
STOP_TOL = 1e-12   # stop tolerance on BOTH sides: coefficient error ~ 30 x tol; 1e-13 is below the FP64
                   # rounding floor of the residual for small lambda
CV_TOL = 1e-5


@pytest.fixture(scope="module")
def tkm():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    import paper_2606_06742_b200 as t
    t.lib()
    return t


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# ------------------------------------------------------------------------------- S1 Gram
@pytest.mark.parametrize("n,p", [(200, 10), (333, 7), (64, 1), (129, 50), (1, 3)])
def test_gram_symmetric(tkm, n, p):
    rng = np.random.default_rng(n + p)
    X = rng.standard_normal((n, p))
    sigma = 1.7 * np.sqrt(p)
    K = tkm.tkm_gram(dev(X), sigma).cpu().numpy()
    Ko = o.gram_rbf(X, sigma)
    assert np.array_equal(K, K.T)                       # bit-exact symmetry
    assert np.all(np.diag(K) == 1.0)
    assert np.max(np.abs(K - Ko) / Ko) < 1e-13


def test_gram_cross_and_strided(tkm):
    import torch
    rng = np.random.default_rng(5)
    A, Bm = rng.standard_normal((150, 12)), rng.standard_normal((77, 12))
    K = tkm.tkm_gram(dev(A), 2.0, dev(Bm)).cpu().numpy()
    assert K.shape == (150, 77)
    assert np.max(np.abs(K - o.gram_rbf(A, 2.0, Bm))) < 1e-14
    wide = torch.zeros((150, 20), dtype=torch.float64, device="cuda")
    wide[:, :12] = dev(A)
    K2 = tkm.tkm_gram(wide[:, :12], 2.0).cpu().numpy()   # ldx = 20 > p
    assert np.max(np.abs(K2 - o.gram_rbf(A, 2.0))) < 1e-14
    Kf = tkm.tkm_gram(dev(A), 2.0, out_dtype=tkm.F32).cpu().numpy()
    assert Kf.dtype == np.float32 and np.array_equal(Kf, o.gram_rbf(A, 2.0).astype(np.float32)) or \
        np.max(np.abs(Kf - o.gram_rbf(A, 2.0))) < 1e-7
    with pytest.raises(tkm.TkmError):
        tkm.tkm_gram(dev(A), 0.0)


# ------------------------------------------------------------------------------- DMMA GEMM
@pytest.mark.parametrize("N,M,K", [(300, 2000, 2000), (37, 130, 70), (64, 64, 16), (1, 5, 3), (130, 257, 1001),
                                   (600, 4096, 512)])
def test_dgemm_nt(tkm, N, M, K):
    rng = np.random.default_rng(N + M + K)
    ldk = (K + 1) // 2 * 2
    P = np.zeros((N, ldk))
    Q = np.zeros((M, ldk))
    P[:, :K] = rng.standard_normal((N, K))
    Q[:, :K] = rng.standard_normal((M, K))
    D = tkm.tkm_dgemm_nt(dev(P)[:, :K], dev(Q)[:, :K]).cpu().numpy()
    ref = P[:, :K] @ Q[:, :K].T
    assert np.max(np.abs(D - ref)) < 1e-13 * K


# ------------------------------------------------------------------------------- S2 spectral setup
def test_spectral_invariants(tkm):
    w = wl.config0(n=333, p=6, seed=4)
    Ko = o.gram_rbf(w.X, w.sigmas[0])
    K = tkm.tkm_gram(dev(w.X), w.sigmas[0])
    spec = tkm.tkm_spectral_setup(K)
    assert (spec.n, spec.r) == (333, 333)
    U = spec.U().cpu().numpy()
    lam, u1 = spec.eigenvalues()
    n = 333
    assert np.max(np.abs(U.T @ U - np.eye(n))) < 1e-12 * n
    assert np.max(np.abs((U * lam) @ U.T - Ko)) < 1e-12 * n
    assert np.all(lam >= 0)
    assert np.max(np.abs(np.sort(lam) - o.spectral_setup(Ko).lam)) < 1e-12 * n
    assert np.max(np.abs(u1 - U.sum(axis=0))) < 1e-12


# ------------------------------------------------------------------------------- S3-S10 full pipeline
def _run_gpu(tkm, w, sigma, foldid, tol, maxit, **kw):
    X, y = dev(w.X), dev(w.y)
    K = tkm.tkm_gram(X, sigma)
    spec = tkm.tkm_spectral_setup(K)
    path = tkm.tkm_fit_path(spec, y, w.loss, w.lambdas, foldid, w.V, tol, maxit, smooth0=w.smooth0, eta=w.eta,
                            rounds=w.rounds, taus=w.taus if len(w.taus) else None, **kw)
    cv = tkm.tkm_exact_cv(path, y, foldid, w.T, w.L, w.V)
    return X, y, spec, path, cv


def _degenerate(w, spec_o, res, c):
    """G18: hinge / check-loss column with no training row strictly inside the quadratic zone (1 - delta, 1 + delta): the
    derivative is locally constant in beta0, so the objective is flat along beta0 on an interval and beta0 (hence
    f and the held-out losses) is not unique; alpha is.  Seen at the largest lambdas of configs[1]."""
    if w.loss not in (o.LOSS_HINGE, o.LOSS_QUANTILE):
        return False
    M = res.cols["M"][:, c] > 0
    f = spec_o.U @ (spec_o.lam * res.a[:, c]) + res.beta0[c]
    d = res.smooth_final if res.smooth_col is None else float(res.smooth_col[c])
    if w.loss == o.LOSS_QUANTILE:      # the same for the check loss: no training residual inside [-gamma, gamma]
        return bool(np.all(np.abs((w.y - f)[M]) >= d))
    u = (w.y * f)[M]
    return bool(np.all((u <= 1 - d) | (u >= 1 + d)))


def _compare_path(tkm, w, sigma, foldid, spec, path, cv, columns=None, coef_tol=COEF_TOL_F64, stop_tol=STOP_TOL,
                  warm_tol=None):
    Ko = o.gram_rbf(w.X, sigma)
    spec_o = o.spectral_setup(Ko)
    res = o.fit_path(spec_o, w.y, w.loss, w.lambdas, foldid, w.V, taus=w.taus, smooth0=w.smooth0, eta=w.eta,
                     rounds=w.rounds, tol=stop_tol, maxit=400000, columns=columns, warm_tol=warm_tol)
    sel = np.arange(res.cols["B"]) if columns is None else np.asarray(columns)
    assert res.flags[sel].sum() == 0
    info = path.info()
    assert info["flags"].sum() == 0, "GPU columns hit maxit"
    U = spec.U().cpu().numpy()
    a_gpu = path.a().cpu().numpy()
    worst = 0.0
    degenerate = set()
    for c in sel:
        alpha_o = spec_o.U @ res.a[:, c]
        alpha_g = U @ a_gpu[c]
        err = np.linalg.norm(alpha_g - alpha_o) / max(np.linalg.norm(alpha_o), 1e-300)
        worst = max(worst, err)
        assert err <= coef_tol, "column %d: relative l2 coefficient error %.3g" % (c, err)
        if _degenerate(w, spec_o, res, c):
            degenerate.add(int(c))
            continue
        assert abs(info["beta0"][c] - res.beta0[c]) <= coef_tol * max(1.0, abs(res.beta0[c])) * 10
    return res, spec_o, worst, degenerate


@pytest.mark.parametrize("name", ["cfg0", "logit_ragged", "kqr_ragged", "hinge_tiny", "dwd_ragged"])
def test_fit_path_and_exact_cv_parity(tkm, name):
    if name == "cfg0":
        w = wl.config0()                                       # BASELINE.json configs[0], full size
    elif name == "logit_ragged":
        w = wl.config2(n=333, p=9, L=7, V=3)
    elif name == "kqr_ragged":
        w = wl.config3(n=261, p=5, L=5, V=4, taus=(0.1, 0.5, 0.9))
    elif name == "dwd_ragged":                                 # DWD (reading G20) on the config-0 generator
        import dataclasses
        w = dataclasses.replace(wl.config0(n=205, p=6, L=6, V=3, seed=17), loss=wl.LOSS_DWD, rounds=1)
    else:
        w = wl.config0(n=37, p=3, L=3, V=2, seed=8)
    # The stop tolerance is an input of both sides (reading G6).  At n = 37, lambda = 1e-4 the oracle's own
    # tol = 1e-12 iterate is 1.5e-10 (relative l2) away from its tol = 1e-14 iterate, i.e. not yet inside
    # the 1e-10 coefficient budget; at 1e-13 it is 1.3e-11.  That case therefore stops at 1e-13.
    stop_tol = 1e-13 if name == "hinge_tiny" else STOP_TOL
    sigma = float(w.sigmas[0])
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    assert np.array_equal(foldid, o.make_folds(w.n, w.V, w.fold_seed))          # bit-exact folds
    X, y, spec, path, cv = _run_gpu(tkm, w, sigma, foldid, stop_tol, 400000)
    res, spec_o, worst, degenerate = _compare_path(tkm, w, sigma, foldid, spec, path, cv, stop_tol=stop_tol)
    print("%s: worst relative l2 coefficient error %.3g" % (name, worst))
    cv_o = o.exact_cv(spec_o, res, w.y, foldid, w.loss, w.taus)
    cv_loss, cv_err, cv_mean, best = cv
    T, L, V = w.T, w.L, w.V
    for t in range(T):
        for l in range(L):
            for v in range(V):
                if (t * (V + 1) + v) * L + l in degenerate:
                    continue
                assert abs(cv_loss[t, l, v] - cv_o[0][t, l, v]) <= CV_TOL
                if w.loss != o.LOSS_QUANTILE:
                    assert cv_err[t, l, v] == cv_o[1][t, l, v]
                else:
                    assert cv_err[t, l, v] == -1
    if not degenerate:
        assert np.max(np.abs(cv_mean - cv_o[2])) <= CV_TOL
        assert np.array_equal(best, cv_o[3])                                     # selected lambda identical
    # reading G22: objective of the non-smoothed problem and its duality-gap certificate, per column
    if w.loss in (o.LOSS_HINGE, o.LOSS_QUANTILE):
        P_o, D_o, gap_o = o.duality_gap(spec_o, res, w.y, w.loss)
        P_g, gap_g = tkm.tkm_path_duality_gap(path, y, foldid)
        keep = np.array([c not in degenerate for c in range(res.cols["B"])])
        assert np.max(np.abs(P_g - P_o)[keep] / np.maximum(1.0, np.abs(P_o[keep]))) <= 1e-9
        assert np.max(np.abs(gap_g - gap_o)[keep]) <= 1e-9 and np.all(gap_g[keep] >= -1e-10)
        assert np.all(gap_g[keep] <= 2 * res.smooth_final)
    else:
        with pytest.raises(tkm.TkmError):
            tkm.tkm_path_duality_gap(path, y, foldid)
    # S10: coefficients and prediction with the selected lambda of variant 0
    l_best = int(cv_o[3][0])
    c = (0 * (V + 1) + V) * L + l_best
    alpha_g, b0_g = tkm.tkm_path_coef(path, 0, l_best, V)
    alpha_o = spec_o.U @ res.a[:, c]
    assert np.linalg.norm(alpha_g.cpu().numpy() - alpha_o) <= COEF_TOL_F64 * np.linalg.norm(alpha_o)
    Xn = wl.new_points(w, 203)
    f_g, lab_g = tkm.tkm_predict(path, 0, l_best, X, dev(Xn), sigma)
    f_o, lab_o = o.predict(w.X, alpha_o, res.beta0[c], sigma, Xn)
    assert np.max(np.abs(f_g.cpu().numpy() - f_o)) <= 1e-9 * max(1.0, np.abs(f_o).max())
    margin = np.min(np.abs(f_o))
    if w.loss != o.LOSS_QUANTILE and margin > 1e-8:
        assert np.array_equal(lab_g.cpu().numpy(), lab_o)                        # labels bit-exact


def _compare_cv_rows(w, foldid, spec_o, res, cv_loss, cols, degenerate):
    L, V = w.L, w.V
    for c in cols:
        t, v, l = c // ((V + 1) * L), (c // L) % (V + 1), c % L
        if v == V or c in degenerate:
            continue
        rows = np.nonzero(foldid == v)[0]
        f = spec_o.U[rows] @ (spec_o.lam * res.a[:, c]) + res.beta0[c]
        tau = float(w.taus[t]) if len(w.taus) else None
        want = np.mean(o.nominal_loss(w.loss, w.y[rows], f, tau))
        assert abs(cv_loss[t, l, v] - want) <= CV_TOL


def test_config1_full_size_bench_configuration(tkm):
    """BASELINE.json configs[1] at full size (n=2000, p=50, 50 lambdas, 5 folds, all 5 sigmas as groups of one
    sweep), in the launch configuration bench.py times (same stop tolerance, warm-start tolerance and delta form).
    Bandwidth index 2 (the median heuristic itself): the oracle (oracle.fit_path, the column-batched mode of the
    same arithmetic, pinned to fit_column in tests/test_oracle_solver.py) fits ALL 300 columns; every coefficient
    vector, the whole CV table, the error counts, the pooled means and the selected lambda are compared.  The
    other four bandwidths: a stated sample of columns."""
    import bench
    w = wl.config1()
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X, y = dev(w.X), dev(w.y)
    specs = [tkm.tkm_spectral_setup(tkm.tkm_gram(X, float(s))) for s in w.sigmas]
    paths = tkm.tkm_fit_path_multi(specs, y, w.loss, w.lambdas, foldid, w.V, bench.STOP_TOL["f64"], bench.MAXIT,
                                   smooth0=w.smooth0, eta=w.eta, rounds=w.rounds, warm_tol=bench.WARM_TOL,
                                   tf32_delta=bench.TF32_DELTA)
    L, V = w.L, w.V
    sample = {2: None, 0: [(5, 35), (0, 10)], 1: [(2, 30)], 3: [(3, 49)], 4: [(1, 45)]}
    for g, vl in sample.items():
        sigma, spec, path = float(w.sigmas[g]), specs[g], paths[g]
        cv = tkm.tkm_exact_cv(path, y, foldid, w.T, w.L, w.V)
        cols = None if vl is None else [v * L + l for (v, l) in vl]
        res, spec_o, worst, degenerate = _compare_path(tkm, w, sigma, foldid, spec, path, cv, columns=cols,
                                                       warm_tol=bench.WARM_TOL)
        print("sigma index %d: %s columns, worst relative l2 coefficient error %.3g"
              % (g, "all" if cols is None else len(cols), worst))
        cv_loss, cv_err, cv_mean, best = cv
        if cols is None:
            cv_o = o.exact_cv(spec_o, res, w.y, foldid, w.loss)
            keep = np.ones((1, L, V), dtype=bool)
            for c in degenerate:
                if (c // L) % (V + 1) < V:
                    keep[0, c % L, (c // L) % (V + 1)] = False
            assert np.max(np.abs(cv_loss - cv_o[0])[keep]) <= CV_TOL
            assert np.array_equal(cv_err[keep], cv_o[1][keep])
            # lambdas with a degenerate hold-out column have a non-unique pooled mean (G18); the others are compared,
            # and the selection is compared when no degenerate lambda is within reach of the minimum on either side
            bad_l = sorted({c % L for c in degenerate if (c // L) % (V + 1) < V})
            ok_l = np.array([l not in bad_l for l in range(L)])
            assert np.max(np.abs(cv_mean - cv_o[2])[0, ok_l]) <= CV_TOL
            order = np.sort(cv_o[2][0])
            print("selected lambda index %d (oracle %d), margin to the runner-up %.3g, degenerate lambdas %s"
                  % (best[0], cv_o[3][0], order[1] - order[0], bad_l))
            reach = min(cv_mean[0, ok_l].min(), cv_o[2][0, ok_l].min()) + 1e-3
            assert all(cv_mean[0, l] > reach and cv_o[2][0, l] > reach for l in bad_l)
            assert np.array_equal(best, cv_o[3])                             # selected lambda identical
        else:
            _compare_cv_rows(w, foldid, spec_o, res, cv_loss, cols, degenerate)
        # properties that hold at any size: every column converged, held-out alpha ~ 0, sum alpha = 0
        info = path.info()
        assert info["flags"].sum() == 0 and np.all(info["kkt"] <= bench.STOP_TOL["f64"])
        U = spec.U().cpu().numpy()
        a_gpu = path.a().cpu().numpy()
        for c in (3, 77, 160, 299):
            v = (c // L) % (V + 1)
            alpha = U @ a_gpu[c]
            sc = np.abs(alpha).max()
            assert abs(alpha.sum()) < 1e-8 * sc * w.n
            if v < V:
                assert np.abs(alpha[foldid == v]).max() < 1e-8 * sc


@pytest.mark.parametrize("cfg,delta", [(2, 0), (2, 2), (3, 0), (3, 2), (3, 3)])
def test_configs_2_3_reduced_n_against_an_oracle_fit(tkm, cfg, delta):
    """BASELINE.json configs[2] (logistic, 100 lambdas, 10 folds) and configs[3] (check loss, tau in {.1,.5,.9}
    stacked on one U, 50 lambdas, 5 folds): their generators, full lambda grids, folds and quantile levels at
    n = 1500, where the oracle can FIT (the full-size runs of tests/test_gpu_fullsize.py are checked against the
    definition only).  configs[2]: all 1100 columns; configs[3]: all tau x all hold-out settings x every fifth
    lambda = 180 of 900 columns (the oracle needs ~1 min for those).  Both sweep precisions the large configs use."""
    w = wl.CONFIGS[cfg](n=1500)
    sigma = float(w.sigmas[0])
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    L, V, T = w.L, w.V, w.T
    cols = None if cfg == 2 else [(t * (V + 1) + v) * L + l for t in range(T) for v in range(V + 1)
                                  for l in range(0, L, 5)]
    # The stop tolerance is an input (reading G6); the comparison target is the minimiser.  On the check-loss columns
    # the oracle's own tol = 1e-12 iterate is 5e-11 .. 8e-11 (relative l2) away from its tol = 1e-14 iterate (condition
    # ~ 70), so two sides that BOTH stop at 1e-12 can be 1.5e-10 apart although each is inside the 1e-10 budget.  The
    # reference therefore stops at 3e-13 here (within 2e-11 of the minimiser; at 1e-13 some of its columns sit on the
    # rounding floor of the residual and never stop); the GPU keeps the 1e-12 of every other test (3e-13 is below
    # the rounding floor of ITS residual on some of these columns).  DESIGN.md section 7.
    X, y, spec, path, cv = _run_gpu(tkm, w, sigma, foldid, STOP_TOL, 400000, warm_tol=1e-3, tf32_delta=delta)
    res, spec_o, worst, degenerate = _compare_path(tkm, w, sigma, foldid, spec, path, cv, columns=cols, warm_tol=1e-3,
                                                   stop_tol=3e-13 if cfg == 3 else STOP_TOL)
    print("cfg %d at n = 1500, tf32_delta %d: worst relative l2 coefficient error %.3g" % (cfg, delta, worst))
    cv_loss, cv_err, cv_mean, best = cv
    if cols is None:
        cv_o = o.exact_cv(spec_o, res, w.y, foldid, w.loss, w.taus)
        assert np.max(np.abs(cv_loss - cv_o[0])) <= CV_TOL and np.array_equal(cv_err, cv_o[1])
        assert np.max(np.abs(cv_mean - cv_o[2])) <= CV_TOL and np.array_equal(best, cv_o[3])
    else:
        _compare_cv_rows(w, foldid, spec_o, res, cv_loss, cols, degenerate)
        # pooled mean of the sampled lambdas (all folds of a sampled lambda are in the sample)
        fsize = np.bincount(foldid, minlength=V).astype(np.float64)
        for t in range(T):
            for l in range(0, L, 5):
                if any((t * (V + 1) + v) * L + l in degenerate for v in range(V)):
                    continue                      # beta0 of a hold-out column is not unique there (G18)
                pooled = 0.0
                for v in range(V):
                    c = (t * (V + 1) + v) * L + l
                    rows = np.nonzero(foldid == v)[0]
                    f = spec_o.U[rows] @ (spec_o.lam * res.a[:, c]) + res.beta0[c]
                    pooled += fsize[v] * np.mean(o.nominal_loss(w.loss, w.y[rows], f, float(w.taus[t])))
                assert abs(cv_mean[t, l] - pooled / w.n) <= CV_TOL


@pytest.mark.parametrize("delta", [0, 2, 3])
def test_config4_parity_set_5000_row_subsample(tkm, delta):
    """BASELINE.json configs[4]: "fp64 oracle on a 5000-row subsample" -- a seeded 5000-row subsample of the
    n = 100000 data set with its own bandwidth (median heuristic on the subsample) and its own m = 1024 landmarks
    (r = 1024 >> the rank-96 thin-U cases above), the full 100-lambda grid; the oracle fits all hold-out settings
    of every twelfth lambda (48 of 600 columns).  Decision values (K~ is only determined to ~1e-9 by the two
    truncated decompositions of reading G11, so coefficients are compared through f), CV losses, error counts."""
    full = wl.config4()
    rows = np.sort(np.random.default_rng(4004).permutation(full.n)[:5000])
    import dataclasses
    Xs = np.ascontiguousarray(full.X[rows])
    w = dataclasses.replace(full, X=Xs, y=full.y[rows].copy(), sigmas=np.array([wl.median_distance(Xs)]),
                            m_landmarks=1024)
    sigma = float(w.sigmas[0])
    idx = wl.landmarks(w.n, w.m_landmarks, w.landmark_seed)
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    L, V = w.L, w.V
    lsel = list(range(4, L, 12))
    cols = [v * L + l for v in range(V + 1) for l in lsel]
    X, y = dev(w.X), dev(w.y)
    spec = tkm.tkm_spectral_setup_nystrom_x(X, sigma, idx)
    spec_o = o.nystrom_setup(w.X, sigma, idx)
    assert spec.r == spec_o.r and spec.r > 900
    path = tkm.tkm_fit_path(spec, y, w.loss, w.lambdas, foldid, V, STOP_TOL, 400000, rounds=w.rounds, warm_tol=1e-3,
                            tf32_delta=delta)
    info = path.info()
    assert info["flags"].sum() == 0
    res = o.fit_path(spec_o, w.y, w.loss, w.lambdas, foldid, V, rounds=w.rounds, tol=STOP_TOL, maxit=400000,
                     columns=cols, warm_tol=1e-3)
    assert res.flags[cols].sum() == 0
    U = spec.U().cpu().numpy()
    lam, _ = spec.eigenvalues()
    a_gpu = path.a().cpu().numpy()
    cv_loss, cv_err, cv_mean, best = tkm.tkm_exact_cv(path, y, foldid, 1, L, V)
    worst = 0.0
    for c in cols:
        v, l = c // L, c % L
        f_o = spec_o.U @ (spec_o.lam * res.a[:, c]) + res.beta0[c]
        f_g = U @ (lam * a_gpu[c]) + info["beta0"][c]
        err = np.max(np.abs(f_g - f_o)) / max(1.0, np.abs(f_o).max())
        worst = max(worst, err)
        assert err < 1e-7, (c, err)
        if v < V:
            r = np.nonzero(foldid == v)[0]
            assert abs(cv_loss[0, l, v] - np.mean(o.nominal_loss(w.loss, w.y[r], f_o[r]))) <= CV_TOL
            margin = np.min(np.abs(f_o[r]))
            if margin > 1e-6:
                assert cv_err[0, l, v] == int(np.sum(o.label_of(f_o[r]) != w.y[r].astype(np.int8)))
    print("configs[4] parity set, tf32_delta %d: worst relative decision-value error %.3g over %d columns"
          % (delta, worst, len(cols)))


@pytest.mark.parametrize("streamed", [False, True])
def test_nystrom_parity(tkm, streamed):
    """streamed: the setup forms K_mm itself and produces K_nm 64 rows at a time (11 blocks, ragged last one)."""
    w = wl.config4(n=700, p=8, m=96, L=5, V=3)
    sigma = float(w.sigmas[0])
    idx = wl.landmarks(w.n, w.m_landmarks, w.landmark_seed)
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X, y = dev(w.X), dev(w.y)
    Xl = X[dev(idx)]
    K_nm = tkm.tkm_gram(X, sigma, Xl)
    K_mm = tkm.tkm_gram(Xl, sigma)
    spec = (tkm.tkm_spectral_setup_nystrom_x(X, sigma, idx, block_rows=64) if streamed
            else tkm.tkm_spectral_setup(nystrom=(K_nm, K_mm, idx)))
    spec_o = o.nystrom_setup(w.X, sigma, idx)
    assert spec.r == spec_o.r
    U = spec.U().cpu().numpy()
    lam, _ = spec.eigenvalues()
    Kt_o = (spec_o.U * spec_o.lam) @ spec_o.U.T
    assert np.max(np.abs((U * lam) @ U.T - Kt_o)) < 1e-9
    path = tkm.tkm_fit_path(spec, y, w.loss, w.lambdas, foldid, w.V, STOP_TOL, 200000, rounds=w.rounds)
    res = o.fit_path(spec_o, w.y, w.loss, w.lambdas, foldid, w.V, rounds=w.rounds, tol=STOP_TOL, maxit=400000)
    a_gpu = path.a().cpu().numpy()
    info = path.info()
    for c in range(res.cols["B"]):
        f_o = spec_o.U @ (spec_o.lam * res.a[:, c]) + res.beta0[c]
        f_g = U @ (lam * a_gpu[c]) + info["beta0"][c]
        assert np.max(np.abs(f_g - f_o)) < 1e-7 * max(1.0, np.abs(f_o).max())
    cv = tkm.tkm_exact_cv(path, y, foldid, 1, w.L, w.V)
    cv_o = o.exact_cv(spec_o, res, w.y, foldid, w.loss)
    assert np.max(np.abs(cv[0] - cv_o[0])) <= CV_TOL and np.array_equal(cv[1], cv_o[1])
    assert np.array_equal(cv[3], cv_o[3])
    l = int(cv_o[3][0])
    c = w.V * w.L + l
    gam_g, b0 = tkm.tkm_path_coef(path, 0, l, w.V)
    gam_o = o.nystrom_landmark_weights(spec_o, res.a[:, c])
    Xn = wl.new_points(w, 64)
    f_g, lab_g = tkm.tkm_predict(path, 0, l, X, dev(Xn), sigma)
    f_o, lab_o = o.predict(w.X[idx], gam_o, res.beta0[c], sigma, Xn)
    assert np.max(np.abs(f_g.cpu().numpy() - f_o)) < 1e-6
    if np.min(np.abs(f_o)) > 1e-6:
        assert np.array_equal(lab_g.cpu().numpy(), lab_o)


def test_nystrom_streamed_error_paths(tkm):
    w = wl.config4(n=120, p=4, m=16, L=2, V=2)
    X = dev(w.X)
    idx = wl.landmarks(w.n, 16, 3)
    for bad in (dict(sigma=0.0), dict(landmark_idx=np.array([0, 120])), dict(landmark_idx=np.array([-1, 3])),
                dict(block_rows=-5)):
        kw = dict(sigma=1.0, landmark_idx=idx, block_rows=0)
        kw.update(bad)
        with pytest.raises(tkm.TkmError):
            tkm.tkm_spectral_setup_nystrom_x(X, kw["sigma"], kw["landmark_idx"], kw["block_rows"])
    one_block = tkm.tkm_spectral_setup_nystrom_x(X, 2.0, idx)                 # block larger than n
    many = tkm.tkm_spectral_setup_nystrom_x(X, 2.0, idx, block_rows=16)      # 8 blocks, ragged tail of 8
    assert one_block.r == many.r
    l1, _ = one_block.eigenvalues()
    l2, _ = many.eigenvalues()
    assert np.max(np.abs(l1 - l2)) <= 1e-12 * l1.max()


# ------------------------------------------------------------------------------- outer control (reading G23)
@pytest.mark.parametrize("loss_name,warm_tol,delta", [("hinge", 0.0, 0), ("hinge", 1e-3, 0), ("hinge", 1e-3, 2),
                                                       ("kqr", 1e-3, 0)])
def test_outer_control_matches_the_oracle(tkm, loss_name, warm_tol, delta):
    """PAPER.md:220-222 under reading G23: with gap_tol > 0 every column leaves the delta-schedule at the first
    level whose solution certifies the duality gap.  The exit level is a decision taken on floating-point gaps, so
    it is compared where the oracle's gap is clear of gap_tol (and the GPU's level must carry a valid certificate
    everywhere); coefficients are compared with the oracle's fixed-schedule fit of the GPU's own level."""
    if loss_name == "hinge":
        w = wl.config0(n=230, p=8, L=9, V=4, seed=41)
    else:
        w = wl.config3(n=190, p=5, L=6, V=3, taus=(0.25, 0.75))
    R, gap_tol = 4, 3e-3
    sigma = float(w.sigmas[0])
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X, y, spec, path, cv = _run_gpu(tkm, w, sigma, foldid, STOP_TOL, 400000, warm_tol=warm_tol, tf32_delta=delta,
                                    gap_tol=gap_tol, delta_min_live=16)
    lev_g, sm_g = path.levels()
    info = path.info()
    assert (info["flags"] & 1).sum() == 0
    spec_o = o.spectral_setup(o.gram_rbf(w.X, sigma))
    kw = dict(taus=w.taus, smooth0=w.smooth0, eta=w.eta, tol=STOP_TOL, maxit=400000)
    res = o.fit_path(spec_o, w.y, w.loss, w.lambdas, foldid, w.V, rounds=R, warm_tol=warm_tol or None, gap_tol=gap_tol,
                     **kw)
    fixed = {k: o.fit_path(spec_o, w.y, w.loss, w.lambdas, foldid, w.V, rounds=k + 1, **kw) for k in range(R)}
    gaps = {k: o.duality_gap(spec_o, fixed[k], w.y, w.loss)[2] for k in range(R)}
    assert len(set(res.level.tolist())) >= 2
    assert np.allclose(sm_g, w.smooth0 * w.eta ** lev_g)
    U = spec.U().cpu().numpy()
    a_gpu = path.a().cpu().numpy()
    P_g, gap_g = tkm.tkm_path_duality_gap(path, y, foldid)
    differ = 0
    for c in range(res.cols["B"]):
        k = int(lev_g[c])
        clear = all(abs(gaps[j][c] - gap_tol) > 0.3 * gap_tol for j in range(R - 1))
        if clear:
            assert k == res.level[c], (c, k, res.level[c])
        differ += k != res.level[c]
        if k < R - 1:
            assert gap_g[c] <= gap_tol + 1e-9 and gaps[k][c] <= gap_tol + 1e-9       # a valid certificate
        else:
            assert bool(info["flags"][c] & 2) == bool(gap_g[c] > gap_tol)
        if _degenerate(w, spec_o, fixed[k], c):
            continue
        assert abs(gap_g[c] - gaps[k][c]) <= 1e-9
        alpha_o, alpha_g = spec_o.U @ fixed[k].a[:, c], U @ a_gpu[c]
        assert np.linalg.norm(alpha_g - alpha_o) <= COEF_TOL_F64 * np.linalg.norm(alpha_o), (c, k)
    print("%s warm_tol %g delta %d: exit levels %s (oracle %s), %d near-threshold columns differ; column-iterations "
          "%d (fixed schedule of %d rounds: oracle %d)" % (loss_name, warm_tol, delta, np.bincount(lev_g, minlength=R),
                                                          np.bincount(res.level, minlength=R), differ,
                                                          path.total_col_iters, R, fixed[R - 1].iters.sum()))


# ------------------------------------------------------------------------------- edge cases / errors
def test_error_paths_and_maxit_flag(tkm):
    w = wl.config0(n=50, p=3, L=2, V=2, seed=3)
    foldid = tkm.tkm_make_folds(w.n, w.V, 1)
    X, y = dev(w.X), dev(w.y)
    spec = tkm.tkm_spectral_setup(tkm.tkm_gram(X, float(w.sigmas[0])))
    with pytest.raises(tkm.TkmError) as e:
        tkm.tkm_fit_path(spec, y, w.loss, [1.0, -1.0], foldid, w.V, 1e-9, 100)
    assert e.value.code == 1
    bad = w.y.copy()
    bad[3] = 0.5
    with pytest.raises(tkm.TkmError):
        tkm.tkm_fit_path(spec, dev(bad), w.loss, w.lambdas, foldid, w.V, 1e-9, 100)
    with pytest.raises(tkm.TkmError):
        tkm.tkm_fit_path(spec, y, w.loss, w.lambdas, np.zeros(w.n, dtype=np.int32), w.V, 1e-9, 100)
    path = tkm.tkm_fit_path(spec, y, w.loss, w.lambdas, foldid, w.V, 1e-13, 3, rounds=2)
    assert path.status == 5 and path.info()["flags"].sum() > 0            # TKM_ENOTCONV, results written
    assert np.all(path.info()["iters"] <= 6)
    # warm start from a converged path converges immediately
    p1 = tkm.tkm_fit_path(spec, y, w.loss, w.lambdas, foldid, w.V, 1e-10, 100000, rounds=1, smooth0=0.125)
    p2 = tkm.tkm_fit_path(spec, y, w.loss, w.lambdas, foldid, w.V, 1e-10, 100000, rounds=1, smooth0=0.125, warm=p1)
    assert p2.info()["iters"].max() <= 2


# ------------------------------------------------------------------------------- grouped sweep / host pipeline
def test_fit_path_multi_matches_oracle_per_group(tkm):
    """tkm_fit_path_multi: three bandwidths swept as groups of one launch; every group must match the oracle
    run on its own Gram matrix (the groups share nothing but y, the folds and the lambda grid)."""
    w = wl.config0(n=150, p=5, L=6, V=3, seed=11)
    sig = [0.5 * float(w.sigmas[0]), float(w.sigmas[0]), 2.0 * float(w.sigmas[0])]
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X, y = dev(w.X), dev(w.y)
    specs = [tkm.tkm_spectral_setup(tkm.tkm_gram(X, s)) for s in sig]
    paths = tkm.tkm_fit_path_multi(specs, y, w.loss, w.lambdas, foldid, w.V, STOP_TOL, 400000, rounds=w.rounds)
    assert len(paths) == 3
    for s, spec, path in zip(sig, specs, paths):
        cv = tkm.tkm_exact_cv(path, y, foldid, w.T, w.L, w.V)
        res, spec_o, worst, degenerate = _compare_path(tkm, w, s, foldid, spec, path, cv)
        cv_o = o.exact_cv(spec_o, res, w.y, foldid, w.loss, w.taus)
        if not degenerate:
            assert np.max(np.abs(cv[0] - cv_o[0])) <= CV_TOL and np.array_equal(cv[1], cv_o[1])
            assert np.array_equal(cv[3], cv_o[3])
    # warm start of all groups from the converged paths: nothing left to do
    again = tkm.tkm_fit_path_multi(specs, y, w.loss, w.lambdas, foldid, w.V, 1e-10, 1000, rounds=1,
                                   smooth0=w.smooth0 * w.eta ** (w.rounds - 1), warm=paths)
    assert max(p.info()["iters"].max() for p in again) <= 2
    with pytest.raises(tkm.TkmError):
        w2 = wl.config0(n=60, p=5, L=6, V=3, seed=11)
        other = tkm.tkm_spectral_setup(tkm.tkm_gram(dev(w2.X), sig[0]))
        tkm.tkm_fit_path_multi([specs[0], other], y, w.loss, w.lambdas, foldid, w.V, STOP_TOL, 100)


@pytest.mark.parametrize("mode", [1, 2, 3])
def test_fit_path_multi_agrees_with_single_calls_in_the_delta_forms(tkm, mode):
    """Groups of one launch against separate tkm_fit_path calls with the delta forms on: tile choice and the
    all-FP64 switch depend on totals over the groups, so the iterates differ -- the minimisers must not
    (include/tkm.h: "same minimiser within tol")."""
    w = wl.config0(n=260, p=5, L=8, V=3, seed=13)
    sig = [0.6 * float(w.sigmas[0]), 1.5 * float(w.sigmas[0])]
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X, y = dev(w.X), dev(w.y)
    specs = [tkm.tkm_spectral_setup(tkm.tkm_gram(X, s)) for s in sig]
    kw = dict(rounds=w.rounds, tf32_delta=mode, delta_min_live=16, profile=1)
    multi = tkm.tkm_fit_path_multi(specs, y, w.loss, w.lambdas, foldid, w.V, STOP_TOL, 400000, **kw)
    assert multi[0].profile()["launches"][3] > 0, "the delta form never engaged"
    for spec, pm in zip(specs, multi):
        ps = tkm.tkm_fit_path(spec, y, w.loss, w.lambdas, foldid, w.V, STOP_TOL, 400000, **kw)
        assert pm.status == 0 and ps.status == 0
        am, as_ = pm.a().cpu().numpy(), ps.a().cpu().numpy()
        U = spec.U().cpu().numpy()
        worst = 0.0
        for c in range(pm.B):
            fm, fs = U @ am[c], U @ as_[c]
            worst = max(worst, np.linalg.norm(fm - fs) / max(np.linalg.norm(fs), 1e-300))
        print("mode %d: multi vs single, worst relative l2 difference of alpha %.3g" % (mode, worst))
        assert worst <= 2 * COEF_TOL_F64      # each side is within COEF_TOL_F64 of the minimiser
        ps.close()


def test_train_tune_host_matches_oracle(tkm):
    """The end-to-end call bench.py times as `e2e`: host buffers in, CV tables and coefficients out."""
    w = wl.config0(n=120, p=4, L=5, V=3, seed=5)
    sig = np.array([float(w.sigmas[0]), 1.7 * float(w.sigmas[0])])
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    r = tkm.tkm_train_tune_host(w.X, w.y, sig, w.loss, w.lambdas, foldid, w.V, STOP_TOL, 400000, rounds=w.rounds)
    assert r["status"] == 0
    for g, s in enumerate(sig):
        so = o.spectral_setup(o.gram_rbf(w.X, s))
        res = o.fit_path(so, w.y, w.loss, w.lambdas, foldid, w.V, rounds=w.rounds, tol=STOP_TOL, maxit=400000)
        cvo = o.exact_cv(so, res, w.y, foldid, w.loss)
        assert np.max(np.abs(r["cv_loss"][g] - cvo[0])) <= CV_TOL
        assert np.array_equal(r["cv_err"][g], cvo[1]) and np.array_equal(r["best_l"][g], cvo[3])
        c = w.V * w.L + int(cvo[3][0])
        alpha_o = so.U @ res.a[:, c]
        assert np.linalg.norm(r["alpha"][g] - alpha_o) <= COEF_TOL_F64 * np.linalg.norm(alpha_o)
        assert abs(r["beta0"][g] - res.beta0[c]) <= 1e-9 * max(1.0, abs(res.beta0[c]))


# ------------------------------------------------------------------------------- tcgen05 3xTF32 contraction
@pytest.mark.parametrize("N,M,K,cfg", [(64, 128, 32, 0), (37, 130, 70, 0), (128, 256, 512, 1), (300, 2000, 2000, -1),
                                       (100, 333, 1001, 2), (700, 520, 256, -1), (513, 128, 64, -1), (5, 1000, 96, -1)])
def test_tf32x3_gemm_nt(tkm, N, M, K, cfg):
    """The tcgen05 (TMEM accumulator) 3xTF32 product against FP64: the error is that of FP32 accumulation in the
    tensor core, which truncates -- it grows like K 2^-24 relative to the size of the partial sums."""
    import torch
    g = torch.Generator(device="cuda").manual_seed(N + M + K)
    P = torch.randn((N, K), device="cuda", dtype=torch.float64, generator=g)
    Q = torch.randn((M, K), device="cuda", dtype=torch.float64, generator=g)
    D = tkm.tkm_tf32x3_gemm_nt(P, Q, cfg=cfg)
    ref = P @ Q.T
    err = float((D - ref).abs().max())
    bound = 4.0 * K * 2.0 ** -24 * float(np.sqrt(K)) + 1e-5      # ~ (K/8 x 3 accumulations) ulps of sqrt(K)-sized sums
    assert err <= bound, (err, bound)
    plain_tf32 = float(np.sqrt(K)) * 2.0 ** -11                   # rms error of a single-TF32 product sum
    assert err < 0.25 * plain_tf32                                # max over all outputs vs that rms


def test_gram_multi_bit_identical_to_single(tkm):
    rng = np.random.default_rng(3)
    X = rng.standard_normal((333, 17))
    sig = [1.1, 2.9, 7.0]
    Ks = tkm.tkm_gram_multi(dev(X), sig)
    for s, K in zip(sig, Ks):
        K1 = tkm.tkm_gram(dev(X), s)
        assert bool((K == K1).all())
        Kn = K.cpu().numpy()
        assert np.array_equal(Kn, Kn.T) and np.all(np.diag(Kn) == 1.0)
        assert np.max(np.abs(Kn - o.gram_rbf(X, s)) / o.gram_rbf(X, s)) < 1e-13
    with pytest.raises(tkm.TkmError):
        tkm.tkm_gram_multi(dev(X), [1.0, 0.0])


def test_leave_one_out_form(tkm):
    """Algorithm 1 in its printed leave-one-out form: V = n folds of one sample each,
    B = L (n + 1) columns.  Every held-out decision value must equal the oracle's."""
    w = wl.config0(n=48, p=4, L=3, V=48, seed=13)
    sigma = float(w.sigmas[0])
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    assert sorted(foldid.tolist()) == list(range(w.n))                       # a permutation: one row per fold
    X, y, spec, path, cv = _run_gpu(tkm, w, sigma, foldid, STOP_TOL, 400000)
    assert path.B == w.L * (w.n + 1)
    res, spec_o, worst, degenerate = _compare_path(tkm, w, sigma, foldid, spec, path, cv)
    cv_o = o.exact_cv(spec_o, res, w.y, foldid, w.loss, w.taus)
    keep = np.ones((1, w.L, w.V), dtype=bool)
    for c in degenerate:
        if (c // w.L) % (w.V + 1) < w.V:
            keep[0, c % w.L, (c // w.L) % (w.V + 1)] = False
    assert np.max(np.abs(cv[0] - cv_o[0])[keep]) <= CV_TOL
    assert np.array_equal(cv[1][keep], cv_o[1][keep])
    if not degenerate:
        assert np.array_equal(cv[3], cv_o[3])


# ------------------------------------------------------------------------------- Platt scaling (reading G21)
def test_platt_on_held_out_decision_values(tkm):
    w = wl.config0(n=260, p=6, L=5, V=4, seed=23)
    sigma = float(w.sigmas[0])
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X, y, spec, path, cv = _run_gpu(tkm, w, sigma, foldid, STOP_TOL, 400000)
    res, spec_o, worst, degenerate = _compare_path(tkm, w, sigma, foldid, spec, path, cv)
    l = int(cv[3][0])
    f_g = tkm.tkm_cv_decision_values(path, 0, l, foldid)
    f_o = o.cv_decision_values(spec_o, res, foldid, 0, l, w.L, w.V)
    assert np.max(np.abs(f_g.cpu().numpy() - f_o)) <= 1e-8 * max(1.0, np.abs(f_o).max())
    A, B, it = tkm.tkm_platt_fit(f_g, y)
    Ao, Bo = o.platt_fit(f_o, w.y)
    p_g = tkm.tkm_platt_proba(f_g, A, B).cpu().numpy()
    assert np.max(np.abs(p_g - o.platt_proba(f_o, Ao, Bo))) <= 1e-6      # same stopping rule on both sides
    assert abs(A - Ao) <= 1e-5 * max(1.0, abs(Ao)) and abs(B - Bo) <= 1e-5 * max(1.0, abs(Bo)) and it >= 1
    # a second, larger and unbalanced score set straight into the fit kernel
    rng = np.random.default_rng(6)
    yy = np.where(rng.random(5003) < 0.3, 1.0, -1.0)
    ff = 0.8 * yy + rng.standard_normal(5003) - 0.4
    A2, B2, _ = tkm.tkm_platt_fit(dev(ff), dev(yy))
    A2o, B2o = o.platt_fit(ff, yy)
    assert np.max(np.abs(o.platt_proba(ff, A2, B2) - o.platt_proba(ff, A2o, B2o))) <= 1e-6


# ------------------------------------------------------------------------------- delta-form GEMM-B (tcgen05)
@pytest.mark.parametrize("mode", [1, 2, 3])
@pytest.mark.parametrize("name", ["cfg0", "kqr_ragged", "logit_ragged"])
def test_delta_form_sweep_keeps_fp64_parity(tkm, name, mode):
    """tkm_loss_opts.tf32_delta: zeta = U^T z (mode 1) and also F = U Lam a (mode 2) advanced by 3xTF32 increments
    on the tcgen05 tensor cores, exact FP64 contractions and stop test on the last iteration of every batch
    (DESIGN.md 12); mode 3: the same with single-TF32 increment products.  Same 1e-10 coefficient bar."""
    w = {"cfg0": lambda: wl.config0(), "kqr_ragged": lambda: wl.config3(n=261, p=5, L=5, V=4, taus=(0.1, 0.5, 0.9)),
         "logit_ragged": lambda: wl.config2(n=333, p=9, L=7, V=3)}[name]()
    sigma = float(w.sigmas[0])
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X, y, spec, path, cv = _run_gpu(tkm, w, sigma, foldid, STOP_TOL, 400000, tf32_delta=mode,
                                    delta_min_live=16, profile=1)   # small n: the cost model alone would stay all-FP64
    if name != "logit_ragged":      # (a handful of batches there: the sampled first iterations may all be exact ones)
        assert path.profile()["launches"][3] > 0 and (mode == 1 or path.profile()["launches"][2] > 0), \
            "the delta form never engaged"
    res, spec_o, worst, degenerate = _compare_path(tkm, w, sigma, foldid, spec, path, cv)
    print("%s (delta form %d): worst relative l2 coefficient error %.3g" % (name, mode, worst))
    cv_o = o.exact_cv(spec_o, res, w.y, foldid, w.loss, w.taus)
    if not degenerate:
        assert np.max(np.abs(cv[0] - cv_o[0])) <= CV_TOL and np.array_equal(cv[3], cv_o[3])


# ----------------------------------------------------------------- column sharding over GPUs
def test_column_sharded_lambda_grid_matches_single_gpu_and_oracle(tkm):
    """The lambda grid interleaved over `world` ranks (here the ranks' shares run one after another on the one
    GPU: they never wait on each other), tables reassembled, lambda selected by tkm_cv_select: identical
    selection, tables equal to the unsharded run's and the oracle's."""
    from paper_2606_06742_b200 import ranks
    w = wl.config0(n=300, p=6, L=7, V=4, seed=31)
    sigma = float(w.sigmas[0])
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X, y, spec, path, cv = _run_gpu(tkm, w, sigma, foldid, STOP_TOL, 400000)
    res, spec_o, worst, degenerate = _compare_path(tkm, w, sigma, foldid, spec, path, cv)
    cv_o = o.exact_cv(spec_o, res, w.y, foldid, w.loss, w.taus)
    fsize = np.bincount(foldid, minlength=w.V).astype(np.float64)
    for world in (2, 3):
        loss_full = np.full((1, w.L, w.V), np.nan)
        err_full = np.full((1, w.L, w.V), -7, dtype=np.int64)
        for rank in range(world):
            mine = ranks.lambda_slice(w.L, rank, world)
            part = tkm.tkm_fit_path(spec, y, w.loss, w.lambdas[mine], foldid, w.V, STOP_TOL, 400000, smooth0=w.smooth0,
                                    eta=w.eta, rounds=w.rounds)
            assert part.info()["flags"].sum() == 0
            l_loss, l_err, _, _ = tkm.tkm_exact_cv(part, y, foldid, 1, len(mine), w.V)
            loss_full[:, mine], err_full[:, mine] = l_loss, l_err
            for j, l in enumerate(mine):      # a sharded column is the same fit as the unsharded one
                a_p, b_p = tkm.tkm_path_coef(part, 0, j, w.V)
                a_f, b_f = tkm.tkm_path_coef(path, 0, int(l), w.V)
                assert float((a_p - a_f).norm() / a_f.norm()) <= 2 * COEF_TOL_F64 and abs(b_p - b_f) <= 1e-9
        cv_mean, best = tkm.tkm_cv_select(loss_full, fsize, w.lambdas)
        assert np.max(np.abs(loss_full - cv[0])) <= 1e-9 and np.array_equal(err_full, cv[1])
        assert np.max(np.abs(loss_full - cv_o[0])) <= CV_TOL and np.array_equal(err_full, cv_o[1])
        assert np.array_equal(best, cv[3]) and np.array_equal(best, cv_o[3])
        assert np.max(np.abs(cv_mean - (loss_full * fsize).sum(axis=2) / w.n)) <= 1e-14
    # world = 1 through the driver itself
    p1, mine, cl, ce, cm, b = tkm.tkm_fit_cv_sharded(spec, y, w.loss, w.lambdas, foldid, w.V, STOP_TOL, 400000,
                                                     smooth0=w.smooth0, eta=w.eta, rounds=w.rounds)
    assert mine.tolist() == list(range(w.L)) and np.array_equal(b, cv[3]) and np.array_equal(ce, cv[1])
    assert np.max(np.abs(cl - cv[0])) <= 1e-9
    # ties -> largest lambda (reading G14): a flat table selects index of max(lambda)
    flat = np.ones((2, w.L, w.V))
    _, bt = tkm.tkm_cv_select(flat, fsize, w.lambdas)
    assert np.all(bt == int(np.argmax(w.lambdas)))
    with pytest.raises(tkm.TkmError):
        tkm.tkm_cv_select(flat, np.zeros(w.V), w.lambdas)


# --------------------------------------------------- K-split GEMM-B (thin U, long contraction)
_KSPLIT_ORACLE = {}


@pytest.mark.parametrize("mode", [0, 2])
def test_thin_u_long_contraction_ksplit_parity(tkm, mode):
    """n = 17000 rows, r <= 48: GEMM-B has one output tile per 54 columns and a 17000-deep contraction, so the
    library cuts K into ranges (FP64 DMMA kernel: mode 0 and the exact iterations; tcgen05 kernel: the delta
    iterations of mode 2) and sums the partials in a fixed order.  Decision values and CV tables against the oracle."""
    w = wl.config4(n=17000, p=6, m=48, L=9, V=5, seed=77)
    w.lambdas[:] = np.logspace(0, -2, 9)
    sigma = float(w.sigmas[0])
    idx = wl.landmarks(w.n, w.m_landmarks, w.landmark_seed)
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X, y = dev(w.X), dev(w.y)
    spec = tkm.tkm_spectral_setup_nystrom_x(X, sigma, idx, block_rows=4096)
    spec_o = o.nystrom_setup(w.X, sigma, idx)
    assert spec.r == spec_o.r
    tol = 1e-11
    path = tkm.tkm_fit_path(spec, y, w.loss, w.lambdas, foldid, w.V, tol, 200000, rounds=w.rounds, tf32_delta=mode,
                            delta_min_live=16, profile=1)
    if mode:
        assert path.profile()["launches"][3] > 0, "the delta form never engaged"
    info = path.info()
    assert info["flags"].sum() == 0 and np.all(info["kkt"] <= tol)
    if "res" not in _KSPLIT_ORACLE:      # the oracle's fit takes most of a minute: once for both modes
        _KSPLIT_ORACLE["res"] = o.fit_path(spec_o, w.y, w.loss, w.lambdas, foldid, w.V, rounds=w.rounds, tol=tol,
                                           maxit=400000)
    res = _KSPLIT_ORACLE["res"]
    U = spec.U().cpu().numpy()
    lam, _ = spec.eigenvalues()
    a_gpu = path.a().cpu().numpy()
    worst = 0.0
    for c in range(res.cols["B"]):
        f_o = spec_o.U @ (spec_o.lam * res.a[:, c]) + res.beta0[c]
        f_g = U @ (lam * a_gpu[c]) + info["beta0"][c]
        worst = max(worst, np.max(np.abs(f_g - f_o)) / max(1.0, np.abs(f_o).max()))
    print("ksplit mode %d: max |f_gpu - f_oracle| %.2e" % (mode, worst))
    assert worst < 1e-7
    cv = tkm.tkm_exact_cv(path, y, foldid, 1, w.L, w.V)
    cv_o = o.exact_cv(spec_o, res, w.y, foldid, w.loss)
    assert np.max(np.abs(cv[0] - cv_o[0])) <= CV_TOL and np.array_equal(cv[1], cv_o[1]) and np.array_equal(cv[3], cv_o[3])


def test_dmma_gemm_is_exact_on_freshly_mapped_operands(tkm):
    """Regression for a pipeline race of gemm_f64_tma_kernel: the consumer warps handed a stage back to the TMA
    producer right after ISSUING their fragment loads, and with a starved ring (first wave of a launch whose Q operand
    is freshly mapped memory, two CTAs per SM) the refill overtook the last loads -- four elements of one fragment
    row came from K-tile kt + STAGES.  Integer-valued operands make every product and sum exact in FP64, so the
    result must EQUAL the reference; P[n][l] = (l // 16)^2 + 1000 n tells a stale K-tile or row apart."""
    import torch
    from paper_2606_06742_b200.api import lib, _check
    N, M, K, ldd = 2048, 32768, 2048, 32768 + 64
    l = torch.arange(K, device="cuda", dtype=torch.float64)
    P = ((l // 16) ** 2).repeat(N, 1).contiguous() + torch.arange(N, device="cuda", dtype=torch.float64)[:, None] * 1000.0
    Q0 = torch.ones((M, K), device="cuda", dtype=torch.float64)
    Q0[:, ::7] = 2.0
    ref = P @ Q0.T
    for rep in range(6):
        # a new allocation for Q and the output on every repetition (the caching allocator is emptied first)
        torch.cuda.empty_cache()
        D = torch.empty((N, ldd), device="cuda", dtype=torch.float64)
        Q = torch.empty((M + 64 * (rep + 1), K), device="cuda", dtype=torch.float64)[:M]
        Q.copy_(Q0)
        torch.cuda.synchronize()
        _check(lib().tkm_dgemm_nt(P.data_ptr(), K, Q.data_ptr(), Q.stride(0), D.data_ptr(), ldd, N, M, K, None))
        torch.cuda.synchronize()
        wrong = int((D[:, :M] != ref).sum())
        assert wrong == 0, "repetition %d: %d wrong elements" % (rep, wrong)
        del D, Q


@pytest.mark.parametrize("mode", [0, 2, 3])
def test_whole_step_is_bitwise_reproducible(tkm, mode):
    """Two passes of the whole hot path on the same inputs -- Gram, concurrent decompositions, grouped sweep with
    its device-side compaction and stream-K partial exchange, exact CV -- must give the SAME BITS: every reduction
    has a fixed order and the schedule depends on device-side counts with a fixed lag, never on host timing."""
    import torch
    w = wl.config1(seed=1001)
    w.sigmas = w.sigmas[1:4]
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X, y = dev(w.X), dev(w.y)

    def one_pass():
        Ks = tkm.tkm_gram_multi(X, w.sigmas)
        specs = tkm.tkm_spectral_setup_multi(Ks)
        Us = [sp.U() for sp in specs]
        paths = tkm.tkm_fit_path_multi(specs, y, w.loss, w.lambdas, foldid, w.V, 1e-11, 200000, smooth0=w.smooth0,
                                       eta=w.eta, rounds=w.rounds, warm_tol=1e-3, tf32_delta=mode)
        out = []
        for K, U, path in zip(Ks, Us, paths):
            info = path.info()
            out.append((K, U, path.a(), info["beta0"], info["iters"], tkm.tkm_exact_cv(path, y, foldid, w.T, w.L, w.V)))
            path.close()
        for sp in specs:
            sp.close()
        return out

    first, second = one_pass(), one_pass()
    for g, (a, b) in enumerate(zip(first, second)):
        assert torch.equal(a[0], b[0]), "Gram matrix of bandwidth %d differs between two passes" % g
        assert torch.equal(a[1], b[1]), "eigenvectors of bandwidth %d differ" % g
        assert torch.equal(a[2], b[2]), "coefficients of bandwidth %d differ" % g
        assert np.array_equal(a[3], b[3]) and np.array_equal(a[4], b[4])
        assert all(np.array_equal(p, q) for p, q in zip(a[5], b[5]))
