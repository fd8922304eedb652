"""paper_2606_06742_b200 -- thin Python binding of libtkm, the B200 (sm_100a) C-ABI library for the
spectral solution path + exact cross-validation of kernel machines (TorchKM, arxiv/paper_2606_06742).

Argument marshalling only: every step of the path (Gram, spectral setup, sweep, exact CV, predict)
runs in the CUDA kernels of `csrc/`, reached through the `tkm_*` entry points declared in
`include/tkm.h`.  PyTorch is used for device memory and streams.  There is no CPU fallback: a
missing `libtkm.so` or a missing GPU raises.
"""
from .api import (  # noqa: F401
    TkmError, LOSS_HINGE, LOSS_LOGISTIC, LOSS_QUANTILE, LOSS_DWD, F32, F64,
    lib, lib_path, tkm_version, tkm_last_error, tkm_make_folds,
    tkm_gram, tkm_gram_multi, tkm_spectral_setup, tkm_spectral_setup_multi, tkm_spectral_setup_nystrom_x, tkm_fit_path, tkm_fit_path_multi, tkm_exact_cv, tkm_cv_select, tkm_path_duality_gap, tkm_fit_cv_sharded, tkm_predict, tkm_predict_noalloc, tkm_path_coef,
    tkm_train_tune_host, tkm_cv_decision_values, tkm_platt_fit, tkm_platt_proba, tkm_dgemm_nt, tkm_gemm_probe, tkm_tf32x3_gemm_nt, tkm_launch_count, tkm_launch_count_reset,
    Spectral, Path, EXPORTED_SYMBOLS,
)
