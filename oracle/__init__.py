"""FP64 CPU oracle for the TorchKM spectral solution path + exact cross-validation.

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s `cpu_baseline` / `--impl reference` legs may import this package.
The product (`paper_2606_06742_b200`, `libtkm.so`) never imports, links or
executes anything in here, and this package never imports the product: the two
share no code.  Plain numpy FP64; written from /root/reference/PAPER.md (cited
as PAPER.md:<line>) with the readings G1..G19 listed in SURVEY.md section 8(c) (G20..G22: DESIGN.md section 3)
and DESIGN.md.

Parity pins (tests/test_oracle_*.py, `-m "not gpu"`):
  gram        two-point closed form, symmetry, unit diagonal, PSD          (P1)
  spectral    U^T U = I, U Lam U^T = K                                      (P2)
  update      dense bordered majoriser solve == spectral step               (P3)
  one-step    huge delta: one step == LS-SVM linear system                  (P4)
  descent     objective non-increasing without momentum                     (P5)
  kkt         alpha = -z/(2 lam), 1^T z = 0, box constraints, dense gradient (P6)
  exact cv    brute-force refit on K[act, act] == masked fit                (P7, P8)
  hinge limit sklearn SVC(kernel="precomputed", C = 1/(2 n lam))            (P9)
  large lam   closed-form intercepts                                        (P10)
  kqr         residual-sign fraction ~ tau                                  (P11)
  path order  alpha^T K alpha monotone along lambda                         (P12)
  nystrom     all points as landmarks == full kernel                        (P13)
  folds       sizes, permutation property, golden bytes from SplitMix64     (P14)
  C <-> lam   objective scaling                                             (P15)
  platt       zero gradient; scikit-learn's _sigmoid_calibration           (P16)
  gap         0 <= gap = O(delta); weak duality; D <= P*(SVC) <= P          (P17)
  outer ctl   gap_tol = 0 == fixed schedule; exit level == first level with gap <= gap_tol; exited column ==
              fixed-schedule fit of that many rounds; P - P*(SVC) <= gap_tol  (P18, reading G23)
Parity unpinned by the paper (inputs, fixed by SURVEY.md 8(c)/DESIGN.md, not
results): delta_0, R, tol, maxit, the t3 noise scale, the landmark seed.
"""
from .gram import gram_rbf
from .spectral import spectral_setup, Spectral
from .losses import psi, curvature, nominal_loss, smooth_loss, LOSS_HINGE, LOSS_LOGISTIC, LOSS_QUANTILE, LOSS_DWD
from .folds import make_folds, splitmix64_stream
from .path import (column_table, column_constants, column_gap, fit_column, fit_path, PathResult,
                   smoothing_levels, path_coef)
from .cv import exact_cv, predict, label_of
from .nystrom import nystrom_setup, nystrom_landmark_weights
from .platt import platt_fit, platt_proba, platt_targets, platt_objective, cv_decision_values
from .refit import brute_force_refit, dense_majoriser, objective
from .diagnostics import duality_gap
