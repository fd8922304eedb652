"""Oracle steps O4-O6: the spectral majorise-minimise solution path (test infrastructure).

Follows PAPER.md Algorithm 1 in its V-fold form
 with the update of PAPER.md:142-146 / 174-176 applied through the
spectral block inverse of PAPER.md:226-230, under the readings of SURVEY.md 8(c):

  G1/G2  bordered majoriser P = [[c n, c 1^T K], [c K 1, 2 lam K + c K^2]], c = curv / n_c;
         P^-1 = (1/s)(1; -v)(1, -v^T) + diag(0, U Pi^-1 U^T) with the Schur complement
         s = c (n - ||u1||^2) + 2 lam c sum_i S_i u1_i^2,  S = Lam Pi^-1 = 1/(2 lam + c Lam)
         (the printed g at PAPER.md:187/230 has lost a minus sign).
  G3     divisor n_c = number of training rows of the column, everywhere.
  G4     r = 1 and (a', b0') = (a, b0) at the start of every smoothing round.
  G6     stop when kkt = max(|gamma0|, n_c ||rho||_2 / sqrt(n)) <= tol.
  G7     fixed smoothing schedule delta_k = delta_0 eta^k, k = 0..R-1, warm-started.
  G10    the fold is a 0/1 mask M on psi (== the zeroed response of PAPER.md:164 for
         margin losses).
  G23    optional outer control of PAPER.md:220-222 ("shrink delta ... until the KKT conditions
         of all SVM models are satisfied"): with gap_tol > 0 a column leaves the smoothing
         schedule after the first round k < R-1 whose solution certifies a duality gap of the
         NON-smoothed problem <= gap_tol (column_gap, reading G22) and keeps that level's
         minimiser.  Rounds before the last may stop at `warm_tol`; such an iterate only screens:
         a column that passes is iterated to `tol` at that level (a fresh round, G4), tested
         again on the converged point, and stays on the schedule if that test fails.
         R stays the cap; gap_tol = 0 is the fixed schedule of G7.

The state is kept in spectral coordinates a = U^T alpha so that K abar = U (Lam * abar)
and every other quantity is elementwise (two contractions with U per iteration,
PAPER.md:232 "O(n^2) matrix-vector multiplications").

Column ordering: c = (t (V+1) + v) L + l;  v = V means "no fold held
out" (the final model for (t, l)).
"""
import dataclasses
import numpy as np

from .losses import psi, curvature, nominal_loss, LOSS_HINGE, LOSS_LOGISTIC, LOSS_QUANTILE, LOSS_DWD


@dataclasses.dataclass
class PathResult:
    a: np.ndarray        # r x B spectral coordinates
    beta0: np.ndarray    # B
    iters: np.ndarray    # B total iterations over all rounds
    kkt: np.ndarray      # B final kkt residual
    flags: np.ndarray    # B, 1 = hit maxit in some round
    cols: dict           # column table (see column_table)
    smooth_final: float  # last delta / gamma of the schedule (None for logistic)
    level: np.ndarray = None       # B, index of the smoothing level each column ended on (R-1 = fixed schedule)
    smooth_col: np.ndarray = None  # B, that level's delta / gamma (nan for the smooth losses)


def smoothing_levels(loss, smooth0, eta, rounds):
    """delta_k (hinge) / gamma_k (quantile) = smooth0 eta^k, k = 0..R-1; logistic: [None].
    PAPER.md:182, 220 (eta = 0.125); reading G7 (fixed R)."""
    if loss in (LOSS_LOGISTIC, LOSS_DWD):
        return [None]
    return [smooth0 * eta ** k for k in range(rounds)]


def column_table(L, V, T, foldid, lambdas, taus):
    """Per-column (t, v, l), lambda, tau, mask M (n x B), n_c."""
    foldid = np.asarray(foldid)
    n = len(foldid)
    B = T * L * (V + 1)
    t_of = np.empty(B, dtype=np.int64)
    v_of = np.empty(B, dtype=np.int64)
    l_of = np.empty(B, dtype=np.int64)
    for t in range(T):
        for v in range(V + 1):
            for l in range(L):
                c = (t * (V + 1) + v) * L + l
                t_of[c], v_of[c], l_of[c] = t, v, l
    M = np.ones((n, B), dtype=np.float64)
    for c in range(B):
        if v_of[c] < V:
            M[foldid == v_of[c], c] = 0.0          # held-out rows: y~ = 0
    n_c = M.sum(axis=0)
    lam_c = np.asarray(lambdas, dtype=np.float64)[l_of]
    tau_c = (np.asarray(taus, dtype=np.float64)[t_of] if len(taus) else np.full(B, np.nan))
    return dict(t=t_of, v=v_of, l=l_of, lam=lam_c, tau=tau_c, M=M, n_c=n_c, L=L, V=V, T=T, B=B)


def column_constants(spec, lam, n_c, curv):
    """O4: c = curv / n_c;  S_i = 1 / (2 lam + c Lam_i);
    s = c (n - ||u1||^2) + 2 lam c sum_i S_i u1_i^2.   (G1)

    For a full orthogonal U, ||u1||^2 = n and the first term is exactly dropped.
    """
    c = curv / n_c
    S = 1.0 / (2.0 * lam + c * spec.lam)
    thin = 0.0 if spec.r == spec.n else (spec.n - float(spec.u1 @ spec.u1))
    s = c * thin + 2.0 * lam * c * float(np.sum(S * spec.u1 * spec.u1))
    return c, S, s


def column_gap(spec, y, loss, a, beta, lam, mask, smooth, tau=None):
    """Duality gap P - D of the NON-smoothed problem at (a, beta) with the dual point the level-`smooth`
    derivative supplies (reading G22; the formulas of oracle/diagnostics.py for one column):
      P = (1/n_c) sum_train loss(y_j, f_j) + lam a^T Lam a,   D = (1/n_c) sum_train (-psi_j) y_j - lam a^T Lam a."""
    f = spec.U @ (spec.lam * a) + beta
    quad = float(np.sum(spec.lam * a * a))
    n_c = float(mask.sum())
    P = float(np.sum(mask * nominal_loss(loss, y, f, tau))) / n_c + lam * quad
    D = float(np.sum(mask * (-psi(loss, y, f, smooth, tau)) * y)) / n_c - lam * quad
    return P - D


def _iterate(spec, y, loss, smooth, lam, mask, tau, a, beta, tol, maxit, restart, momentum, trace, rnd):
    """One smoothing round of O5 for one column from (a, beta): returns (a, beta, iterations, kkt, converged)."""
    U, Lam, u1 = spec.U, spec.lam, spec.u1
    n = spec.n
    n_c = float(mask.sum())
    curv = curvature(loss, smooth)
    c, S, s = column_constants(spec, lam, n_c, curv)
    a_prev, beta_prev, rk = a.copy(), beta, 1.0             # G4
    kkt = np.inf
    for it in range(maxit):
        # 1. Nesterov extrapolation, PAPER.md:199-203 (Alg. 1 l.12-14)
        rk_new = 0.5 * (1.0 + np.sqrt(1.0 + 4.0 * rk * rk))
        mu = (rk - 1.0) / rk_new if momentum else 0.0
        abar = a + mu * (a - a_prev)
        bbar = beta + mu * (beta - beta_prev)
        if trace is not None:
            trace.append((rnd, it, abar.copy(), bbar))
        # 2. zbar, PAPER.md:204 (Alg. 1 l.15); divisor n_c (G3)
        f = U @ (Lam * abar) + bbar
        z = mask * psi(loss, y, f, smooth, tau) / n_c
        gamma0 = float(z.sum())
        # 3. H^-1 d right to left
        rho = U.T @ z + 2.0 * lam * abar
        q = gamma0 - c * float(np.sum(S * Lam * u1 * rho))
        dbeta = q / s
        da = S * (rho - dbeta * c * u1)
        # 4. PAPER.md:210-212 (Alg. 1 l.18-19)
        a_new = abar - da
        beta_new = bbar - dbeta
        if restart and (float(da @ (a_new - a)) + dbeta * (beta_new - beta) > 0.0):
            rk_new = 1.0                                    # gradient restart (not in the paper;
        a_prev, beta_prev = a, beta                         #  does not move the fixed point)
        a, beta, rk = a_new, beta_new, rk_new
        # 5. stop test (G6)
        kkt = max(abs(gamma0), n_c * float(np.sqrt(rho @ rho)) / np.sqrt(n))
        if kkt <= tol:
            return a, beta, it + 1, kkt, True
    return a, beta, maxit, kkt, False


def fit_column(spec, y, loss, levels, lam, mask, tau=None, tol=1e-12, maxit=20000,
               restart=True, a0=None, b0=0.0, momentum=True, trace=None, warm_tol=None, gap_tol=0.0,
               want_level=False):
    """O5/O6 for ONE column: plain loop, mat-vecs with U.  Returns (a, beta0, iters, kkt, flag)
    (+ the index of the level the column ended on when `want_level`).

    `trace`, if a list, receives (round, iteration, abar, bbar) tuples before each update
    (used by the descent pin).  `warm_tol`: stop tolerance of the rounds before the last (None: tol).
    `gap_tol` > 0: the outer control of reading G23.
    """
    r = spec.r
    y = np.asarray(y, dtype=np.float64)
    a = np.zeros(r) if a0 is None else np.array(a0, dtype=np.float64)
    beta = float(b0)
    total_it, flag, kkt, level = 0, 0, np.inf, len(levels) - 1
    for rnd, smooth in enumerate(levels):                   # O6 / PAPER.md:220-222
        last = rnd == len(levels) - 1
        rtol = tol if (last or warm_tol is None) else warm_tol
        a, beta, it, kkt, ok = _iterate(spec, y, loss, smooth, lam, mask, tau, a, beta, rtol, maxit, restart,
                                        momentum, trace, rnd)
        total_it += it
        if not ok:
            flag = 1
        if last or not (gap_tol > 0.0) or smooth is None:
            continue
        if column_gap(spec, y, loss, a, beta, lam, mask, smooth, tau) <= gap_tol:      # G23
            if rtol > tol:
                # the warm iterate only screens: finish this level to the stop tolerance and test the certificate
                # on the converged point (whose dual point is feasible to `tol`)
                a, beta, it, kkt, ok = _iterate(spec, y, loss, smooth, lam, mask, tau, a, beta, tol, maxit,
                                                restart, momentum, trace, rnd)
                total_it += it
                if not ok:
                    flag = 1
                if column_gap(spec, y, loss, a, beta, lam, mask, smooth, tau) > gap_tol:
                    continue                                # stays on the schedule, warm-started from here
            level = rnd
            break
    if want_level:
        return a, beta, total_it, kkt, flag, level
    return a, beta, total_it, kkt, flag


def fit_path(spec, y, loss, lambdas, foldid, V, taus=(), smooth0=1.0, eta=0.125, rounds=4,
             tol=1e-12, maxit=20000, restart=True, columns=None, warm_tol=None, gap_tol=0.0):
    """All B = T L (V+1) columns.  Same arithmetic as fit_column with a column axis:
    the two contractions become U @ W and U.T @ Z over the still-active columns.

    `columns`: optional list of column indices to fit (others are left at zero and
    flagged 2) -- used to fit a stated subsample at the large configs.
    `warm_tol`, `gap_tol`: as in fit_column (stop tolerance of the warm-start rounds; reading G23).
    """
    U, Lam, u1 = spec.U, spec.lam, spec.u1
    n, r = spec.n, spec.r
    y = np.asarray(y, dtype=np.float64)
    taus = np.asarray(taus, dtype=np.float64)
    T = max(1, len(taus))
    L = len(lambdas)
    cols = column_table(L, V, T, foldid, lambdas, taus)
    B = cols["B"]
    sel = np.arange(B) if columns is None else np.asarray(columns, dtype=np.int64)
    a = np.zeros((r, B))
    beta = np.zeros(B)
    iters = np.zeros(B, dtype=np.int64)
    kkt = np.full(B, np.inf)
    flags = np.zeros(B, dtype=np.int32)
    if columns is not None:
        flags[:] = 2
        flags[sel] = 0
    levels = smoothing_levels(loss, smooth0, eta, rounds)
    level = np.full(B, len(levels) - 1, dtype=np.int64)
    lam_c, n_c, M, tau_c = cols["lam"], cols["n_c"], cols["M"], cols["tau"]
    thin = 0.0 if r == n else (n - float(u1 @ u1))

    def run_round(smooth, start, rtol):
        """One smoothing round (G4: fresh momentum) of the columns `start`, each until kkt <= rtol."""
        curv = curvature(loss, smooth)
        c = curv / n_c                                             # B
        S = 1.0 / (2.0 * lam_c[None, :] + c[None, :] * Lam[:, None])   # r x B
        s = c * thin + 2.0 * lam_c * c * np.sum(S * (u1 * u1)[:, None], axis=0)
        a_prev = a.copy()
        beta_prev = beta.copy()
        rk = np.ones(B)
        act = start.copy()
        for it in range(maxit):
            if act.size == 0:
                break
            j = act
            rk_new = 0.5 * (1.0 + np.sqrt(1.0 + 4.0 * rk[j] ** 2))
            mu = (rk[j] - 1.0) / rk_new
            abar = a[:, j] + mu * (a[:, j] - a_prev[:, j])
            bbar = beta[j] + mu * (beta[j] - beta_prev[j])
            F = U @ (Lam[:, None] * abar) + bbar[None, :]
            tau_j = tau_c[j][None, :] if loss == LOSS_QUANTILE else None
            Z = M[:, j] * psi(loss, y[:, None], F, smooth, tau_j) / n_c[j][None, :]
            gamma0 = Z.sum(axis=0)
            rho = U.T @ Z + 2.0 * lam_c[j][None, :] * abar
            Sj = S[:, j]
            q = gamma0 - c[j] * np.sum(Sj * (Lam * u1)[:, None] * rho, axis=0)
            dbeta = q / s[j]
            da = Sj * (rho - (dbeta * c[j])[None, :] * u1[:, None])
            a_new = abar - da
            beta_new = bbar - dbeta
            if restart:
                g = np.sum(da * (a_new - a[:, j]), axis=0) + dbeta * (beta_new - beta[j])
                rk_new = np.where(g > 0.0, 1.0, rk_new)
            a_prev[:, j] = a[:, j]
            beta_prev[j] = beta[j]
            a[:, j] = a_new
            beta[j] = beta_new
            rk[j] = rk_new
            iters[j] += 1
            kk = np.maximum(np.abs(gamma0), n_c[j] * np.sqrt(np.sum(rho * rho, axis=0)) / np.sqrt(n))
            kkt[j] = kk
            act = j[kk > rtol]
        flags[act] = 1

    live = sel.copy()                                              # columns still on the schedule
    for rnd, smooth in enumerate(levels):
        last = rnd == len(levels) - 1
        rtol = tol if (last or warm_tol is None) else warm_tol
        run_round(smooth, live, rtol)
        if last or not (gap_tol > 0.0) or smooth is None:
            continue
        def certified(cands):                                      # G23: gap of the non-smoothed problem
            out = []
            for c_ in cands:
                tau = float(tau_c[c_]) if loss == LOSS_QUANTILE else None
                if column_gap(spec, y, loss, a[:, c_], beta[c_], lam_c[c_], M[:, c_], smooth, tau) <= gap_tol:
                    out.append(c_)
            return np.asarray(out, dtype=np.int64)

        passed = certified(live)
        if passed.size and rtol > tol:
            run_round(smooth, passed, tol)                         # the warm iterate only screens: finish the level
            passed = certified(passed)                             # and test the certificate on the converged point
        if passed.size:
            level[passed] = rnd
            live = np.setdiff1d(live, passed)
    smooth_col = np.array([np.nan if levels[k] is None else levels[k] for k in level])
    return PathResult(a=a, beta0=beta, iters=iters, kkt=kkt, flags=flags, cols=cols,
                      smooth_final=levels[-1], level=level, smooth_col=smooth_col)


def path_coef(spec, res, c):
    """O8: alpha = U a (full kernel).  For Nystrom use nystrom_landmark_weights."""
    return spec.U @ res.a[:, c], float(res.beta0[c])
