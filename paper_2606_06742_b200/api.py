"""ctypes binding of libtkm.so: same names as the C ABI (include/tkm.h), torch tensors for [dev]
arguments, numpy arrays for [host] arguments.  No arithmetic of the method lives here."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

LOSS_HINGE, LOSS_LOGISTIC, LOSS_QUANTILE, LOSS_DWD = 0, 1, 2, 3
F32, F64 = 0, 1
TKM_OK, TKM_ENOTCONV = 0, 5

EXPORTED_SYMBOLS = [
    "tkm_gram", "tkm_gram_multi", "tkm_spectral_setup", "tkm_spectral_setup_multi", "tkm_spectral_setup_nystrom_x", "tkm_spectral_free", "tkm_spectral_info", "tkm_spectral_get_u",
    "tkm_fit_path", "tkm_fit_path_multi", "tkm_path_free", "tkm_path_info", "tkm_path_shape", "tkm_path_levels", "tkm_fold_sizes", "tkm_path_profile", "tkm_path_get_a", "tkm_exact_cv", "tkm_cv_select", "tkm_path_duality_gap", "tkm_path_coef",
    "tkm_predict", "tkm_predict_noalloc", "tkm_cv_decision_values", "tkm_platt_fit", "tkm_platt_proba", "tkm_train_tune_host", "tkm_make_folds", "tkm_launch_count", "tkm_launch_count_reset",
    "tkm_dgemm_nt", "tkm_gemm_probe", "tkm_tf32x3_gemm_nt", "tkm_version", "tkm_last_error",
]


class TkmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libtkm error %d: %s" % (code, msg))
        self.code = code


class _LossOpts(C.Structure):
    _fields_ = [("smooth0", C.c_double), ("eta", C.c_double), ("rounds", C.c_int32), ("T", C.c_int32),
                ("taus", C.POINTER(C.c_double)), ("restart", C.c_int32), ("check_every", C.c_int32),
                ("warm_tol", C.c_double), ("profile", C.c_int32), ("tf32_delta", C.c_int32),
                ("gap_tol", C.c_double), ("delta_min_live", C.c_int32)]


class _Nystrom(C.Structure):
    _fields_ = [("K_nm", C.c_void_p), ("ld_nm", C.c_int64), ("K_mm", C.c_void_p), ("ld_mm", C.c_int64),
                ("m", C.c_int64), ("landmark_idx", C.POINTER(C.c_int64))]


def lib_path() -> str:
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), "libtkm.so")


_lib = None


def lib():
    """Loads libtkm.so (built by `python -m paper_2606_06742_b200.build`); raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise TkmError(-1, "%s not found: build it with `python -m paper_2606_06742_b200.build` "
                           "(there is no CPU fallback)" % path)
    L = C.CDLL(path)
    vp, i64, i32, dbl = C.c_void_p, C.c_int64, C.c_int32, C.c_double
    L.tkm_gram.argtypes = [vp, i64, i64, i64, vp, i64, i64, dbl, C.c_int, vp, i64, vp]
    L.tkm_gram_multi.argtypes = [vp, i64, i64, i64, vp, i64, i64, vp, i32, C.c_int, C.POINTER(vp), i64, vp]
    L.tkm_spectral_setup.argtypes = [vp, i64, i64, C.POINTER(_Nystrom), C.POINTER(vp), vp]
    L.tkm_spectral_setup_multi.argtypes = [C.POINTER(vp), i32, i64, i64, C.POINTER(vp), vp]
    L.tkm_spectral_setup_nystrom_x.argtypes = [vp, i64, i64, i64, dbl, vp, i64, i64, C.POINTER(vp), vp]
    L.tkm_spectral_free.argtypes = [vp]
    L.tkm_spectral_free.restype = None
    L.tkm_spectral_info.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), vp, vp]
    L.tkm_spectral_get_u.argtypes = [vp, vp, vp]
    L.tkm_fit_path.argtypes = [vp, vp, C.c_int, C.POINTER(_LossOpts), vp, i32, vp, i32, dbl, i32, vp,
                               C.POINTER(vp), vp]
    L.tkm_fit_path_multi.argtypes = [C.POINTER(vp), i32, vp, C.c_int, C.POINTER(_LossOpts), vp, i32, vp, i32, dbl, i32,
                                     C.POINTER(vp), C.POINTER(vp), vp]
    L.tkm_path_free.argtypes = [vp]
    L.tkm_path_free.restype = None
    L.tkm_path_info.argtypes = [vp, C.POINTER(i32), C.POINTER(i64), vp, vp, vp, vp, C.POINTER(i64)]
    L.tkm_path_levels.argtypes = [vp, vp, vp]
    L.tkm_path_profile.argtypes = [vp, vp, vp, vp]
    L.tkm_path_get_a.argtypes = [vp, vp, vp]
    L.tkm_exact_cv.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
    L.tkm_path_duality_gap.argtypes = [vp, vp, vp, vp, vp, vp]
    L.tkm_cv_select.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp, vp]
    L.tkm_path_coef.argtypes = [vp, i32, i32, i32, vp, C.POINTER(dbl), vp]
    L.tkm_predict.argtypes = [vp, i32, i32, vp, i64, vp, i64, i64, i64, dbl, vp, vp, vp]
    L.tkm_predict_noalloc.argtypes = [vp, i32, i32, vp, i64, vp, i64, i64, i64, dbl, vp, vp, vp]
    L.tkm_cv_decision_values.argtypes = [vp, i32, i32, vp, vp, vp]
    L.tkm_platt_fit.argtypes = [vp, vp, i64, C.POINTER(dbl), C.POINTER(dbl), C.POINTER(i32), vp]
    L.tkm_platt_proba.argtypes = [vp, i64, dbl, dbl, vp, vp]
    L.tkm_train_tune_host.argtypes = [vp, i64, i64, vp, vp, i32, C.c_int, C.POINTER(_LossOpts), vp, i32, vp, i32,
                                      dbl, i32, vp, vp, vp, vp, vp, vp, vp, vp]
    L.tkm_path_shape.argtypes = [vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), C.POINTER(i64)]
    L.tkm_fold_sizes.argtypes = [vp, i64, i32, vp]
    L.tkm_make_folds.argtypes = [i64, i32, C.c_uint64, vp]
    L.tkm_launch_count.restype = i64
    L.tkm_launch_count_reset.restype = None
    L.tkm_dgemm_nt.argtypes = [vp, i64, vp, i64, vp, i64, i64, i64, i64, vp]
    L.tkm_tf32x3_gemm_nt.argtypes = [vp, i64, vp, i64, vp, i64, i64, i64, i64, i32, i32, C.POINTER(C.c_float), vp]
    L.tkm_gemm_probe.argtypes = [i32, i32, i32, i32, i32, i32, C.POINTER(C.c_float), vp]
    L.tkm_last_error.restype = C.c_char_p
    for name in EXPORTED_SYMBOLS:
        getattr(L, name)   # AttributeError if the library does not export a declared symbol
    _lib = L
    return L


def _check(rc, allow_notconv=False):
    if rc == TKM_OK or (allow_notconv and rc == TKM_ENOTCONV):
        return rc
    raise TkmError(rc, lib().tkm_last_error().decode())


def _stream(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dev_f64(t, name):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64):
        raise TypeError("%s must be a CUDA float64 tensor" % name)
    return t


def _host(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def _dev_vec(t, n, name):
    """A contiguous CUDA float64 vector of length n."""
    t = _dev_f64(t, name)
    if t.dim() != 1 or t.numel() != n or (n > 1 and t.stride(0) != 1):
        raise ValueError("%s must be a contiguous vector of length %d" % (name, n))
    return t


def _fold_vec(foldid, n, V):
    fid = _host(foldid, np.int32)
    if fid.shape != (n,):
        raise ValueError("foldid must have length n = %d" % n)
    if n and (fid.min() < 0 or fid.max() >= V):
        raise ValueError("foldid values must lie in [0, V)")
    return fid


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def tkm_version() -> int:
    return lib().tkm_version()


def tkm_last_error() -> str:
    return lib().tkm_last_error().decode()


def tkm_launch_count() -> int:
    return int(lib().tkm_launch_count())


def tkm_launch_count_reset() -> None:
    lib().tkm_launch_count_reset()


def tkm_make_folds(n: int, V: int, seed: int) -> np.ndarray:
    out = np.empty(n, dtype=np.int32)
    _check(lib().tkm_make_folds(n, V, C.c_uint64(seed & (2 ** 64 - 1)), _ptr(out)))
    return out


def tkm_gram(X, sigma: float, X2=None, out_dtype=F64, stream=None):
    """K = exp(-||x_i - x'_j||^2 / (2 sigma^2)); X, X2 CUDA float64 2-D tensors (row stride = ld)."""
    import torch
    X = _dev_f64(X, "X")
    if X.dim() != 2 or X.stride(1) != 1:
        raise ValueError("X must be 2-D with unit inner stride")
    n, p = X.shape
    if X2 is not None:
        X2 = _dev_f64(X2, "X2")
        if X2.dim() != 2 or X2.stride(1) != 1 or X2.shape[1] != p:
            raise ValueError("X2 must be n2 x p with unit inner stride")
        n2, ld2, p2 = X2.shape[0], X2.stride(0), C.c_void_p(X2.data_ptr())
    else:
        n2, ld2, p2 = 0, 0, None
    K = torch.empty((n, n2 if X2 is not None else n), device=X.device,
                    dtype=torch.float64 if out_dtype == F64 else torch.float32)
    _check(lib().tkm_gram(X.data_ptr(), n, p, X.stride(0), p2, n2, ld2, float(sigma), out_dtype,
                          K.data_ptr(), K.stride(0), _stream(stream)))
    return K


def tkm_gram_multi(X, sigmas, out_dtype=F64, stream=None):
    """G symmetric Gram matrices of X (one per bandwidth) from one pass over the squared distances."""
    import torch
    X = _dev_f64(X, "X")
    if X.dim() != 2 or X.stride(1) != 1:
        raise ValueError("X must be 2-D with unit inner stride")
    n, p = X.shape
    sig = _host(np.atleast_1d(sigmas), np.float64)
    G = len(sig)
    Ks = [torch.empty((n, n), device=X.device, dtype=torch.float64 if out_dtype == F64 else torch.float32)
          for _ in range(G)]
    hk = (C.c_void_p * G)(*[K.data_ptr() for K in Ks])
    _check(lib().tkm_gram_multi(X.data_ptr(), n, p, X.stride(0), None, 0, 0, _ptr(sig), G, out_dtype, hk, n,
                                _stream(stream)))
    return Ks


class Spectral:
    """Owner of a tkm_spectral* (freed on garbage collection)."""

    def __init__(self, handle, keepalive=()):
        self._h = handle
        self._keep = keepalive
        n, r = C.c_int64(), C.c_int64()
        _check(lib().tkm_spectral_info(self._h, C.byref(n), C.byref(r), None, None))
        self.n, self.r = n.value, r.value

    def eigenvalues(self):
        lam, u1 = np.empty(self.r), np.empty(self.r)
        _check(lib().tkm_spectral_info(self._h, None, None, _ptr(lam), _ptr(u1)))
        return lam, u1

    def U(self, stream=None):
        import torch
        out = torch.empty((self.n, self.r), device="cuda", dtype=torch.float64)
        _check(lib().tkm_spectral_get_u(self._h, out.data_ptr(), _stream(stream)))
        return out

    def close(self):
        if self._h:
            lib().tkm_spectral_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def tkm_spectral_setup(K=None, n=None, nystrom=None, stream=None) -> Spectral:
    """Full kernel: K (n x n CUDA float64).  Nystrom: nystrom=(K_nm, K_mm, landmark_idx), n = rows."""
    h = C.c_void_p()
    if nystrom is None:
        K = _dev_f64(K, "K")
        n = K.shape[0]
        _check(lib().tkm_spectral_setup(K.data_ptr(), n, K.stride(0), None, C.byref(h), _stream(stream)))
        return Spectral(h)
    K_nm, K_mm, idx = nystrom
    K_nm, K_mm = _dev_f64(K_nm, "K_nm"), _dev_f64(K_mm, "K_mm")
    idx = _host(idx, np.int64)
    ny = _Nystrom(K_nm.data_ptr(), K_nm.stride(0), K_mm.data_ptr(), K_mm.stride(0), K_mm.shape[0],
                  idx.ctypes.data_as(C.POINTER(C.c_int64)))
    _check(lib().tkm_spectral_setup(None, K_nm.shape[0], 0, C.byref(ny), C.byref(h), _stream(stream)))
    return Spectral(h)


def tkm_spectral_setup_nystrom_x(X, sigma: float, landmark_idx, block_rows: int = 0, stream=None) -> Spectral:
    """Nystrom setup from the training matrix itself: K_nm is produced and consumed block_rows rows at a time."""
    X = _dev_f64(X, "X")
    idx = _host(landmark_idx, np.int64)
    h = C.c_void_p()
    _check(lib().tkm_spectral_setup_nystrom_x(X.data_ptr(), X.shape[0], X.shape[1], X.stride(0), float(sigma), _ptr(idx),
                                              len(idx), int(block_rows), C.byref(h), _stream(stream)))
    return Spectral(h, keepalive=(idx,))


def tkm_spectral_setup_multi(Ks, stream=None):
    """Concurrent full-kernel setups of G Gram matrices of one size -> list of G Spectral handles."""
    Ks = [_dev_f64(K, "K") for K in Ks]
    G, n, ld = len(Ks), Ks[0].shape[0], Ks[0].stride(0)
    if any(K.shape != (n, n) or K.stride(0) != ld or K.stride(1) != 1 for K in Ks):
        raise ValueError("all K must be n x n with the same row stride")
    hk = (C.c_void_p * G)(*[K.data_ptr() for K in Ks])
    ho = (C.c_void_p * G)()
    _check(lib().tkm_spectral_setup_multi(hk, G, n, ld, ho, _stream(stream)))
    return [Spectral(C.c_void_p(ho[g])) for g in range(G)]


class Path:
    """Owner of a tkm_path*; keeps its Spectral alive."""

    def __init__(self, handle, spec, status):
        self._h = handle
        self.spec = spec
        self.status = status            # TKM_OK or TKM_ENOTCONV
        B, r, tot = C.c_int32(), C.c_int64(), C.c_int64()
        _check(lib().tkm_path_info(self._h, C.byref(B), C.byref(r), None, None, None, None, C.byref(tot)))
        self.B, self.r, self.total_col_iters = B.value, r.value, tot.value
        T, L, V, n = C.c_int32(), C.c_int32(), C.c_int32(), C.c_int64()
        _check(lib().tkm_path_shape(self._h, C.byref(T), C.byref(L), C.byref(V), C.byref(n)))
        self.T, self.L, self.V, self.n = T.value, L.value, V.value, n.value

    def info(self):
        iters = np.empty(self.B, dtype=np.int32)
        kkt = np.empty(self.B)
        flags = np.empty(self.B, dtype=np.int32)
        beta0 = np.empty(self.B)
        _check(lib().tkm_path_info(self._h, None, None, _ptr(iters), _ptr(kkt), _ptr(flags), _ptr(beta0), None))
        return dict(iters=iters, kkt=kkt, flags=flags, beta0=beta0)

    def levels(self):
        """(level index, smoothing parameter) every column ended on (reading G23)."""
        lev, sm = np.empty(self.B, dtype=np.int32), np.empty(self.B)
        _check(lib().tkm_path_levels(self._h, _ptr(lev), _ptr(sm)))
        return lev, sm

    def profile(self):
        """Sampled launches by family: index 0/1 = FP64 DMMA GEMM-A/B, 2/3 = tcgen05 3xTF32 delta GEMM-A/B."""
        ms, fl = np.zeros(4), np.zeros(4)
        nl = np.zeros(4, dtype=np.int64)
        _check(lib().tkm_path_profile(self._h, _ptr(ms), _ptr(fl), _ptr(nl)))
        return dict(ms=ms, flops=fl, launches=nl)

    def a(self, stream=None):
        import torch
        out = torch.empty((self.B, self.r), device="cuda", dtype=torch.float64)
        _check(lib().tkm_path_get_a(self._h, out.data_ptr(), _stream(stream)))
        return out

    def close(self):
        if self._h:
            lib().tkm_path_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _opts(loss, smooth0, eta, rounds, taus, restart, check_every, warm_tol, profile=False, tf32_delta=0, gap_tol=0.0,
          delta_min_live=0):
    taus_arr = _host(taus if taus is not None else [], np.float64)
    o = _LossOpts(float(smooth0), float(eta), int(rounds), int(len(taus_arr)),
                  taus_arr.ctypes.data_as(C.POINTER(C.c_double)) if len(taus_arr) else None,
                  int(bool(restart)), int(check_every), float(warm_tol), int(profile), int(tf32_delta), float(gap_tol),
                  int(delta_min_live))
    return o, taus_arr


def tkm_fit_path(spec: Spectral, y, loss: int, lambdas, foldid, V: int, tol: float, maxit: int,
                 smooth0=1.0, eta=0.125, rounds=4, taus=None, restart=True, check_every=0, warm_tol=0.0,
                 warm: Path | None = None, profile=False, tf32_delta=0, gap_tol=0.0, delta_min_live=0, stream=None) -> Path:
    y = _dev_vec(y, spec.n, "y")
    lam = _host(lambdas, np.float64)
    fid = _fold_vec(foldid, spec.n, V)
    o, keep = _opts(loss, smooth0, eta, rounds, taus, restart, check_every, warm_tol, profile, tf32_delta, gap_tol,
                    delta_min_live)
    h = C.c_void_p()
    rc = lib().tkm_fit_path(spec._h, y.data_ptr(), loss, C.byref(o), _ptr(lam), len(lam), _ptr(fid), V,
                            float(tol), int(maxit), warm._h if warm is not None else None, C.byref(h),
                            _stream(stream))
    _check(rc, allow_notconv=True)
    return Path(h, spec, rc)


def tkm_fit_path_multi(specs, y, loss: int, lambdas, foldid, V: int, tol: float, maxit: int,
                       smooth0=1.0, eta=0.125, rounds=4, taus=None, restart=True, check_every=0, warm_tol=0.0,
                       warm=None, profile=False, tf32_delta=0, gap_tol=0.0, delta_min_live=0, stream=None):
    """One sweep over G spectral handles that share y, folds and the lambda grid -> list of G Paths."""
    y = _dev_vec(y, specs[0].n, "y")
    lam = _host(lambdas, np.float64)
    fid = _fold_vec(foldid, specs[0].n, V)
    o, keep = _opts(loss, smooth0, eta, rounds, taus, restart, check_every, warm_tol, profile, tf32_delta, gap_tol,
                    delta_min_live)
    G = len(specs)
    hs = (C.c_void_p * G)(*[s._h for s in specs])
    hw = (C.c_void_p * G)(*[w._h for w in warm]) if warm is not None else None
    ho = (C.c_void_p * G)()
    rc = lib().tkm_fit_path_multi(hs, G, y.data_ptr(), loss, C.byref(o), _ptr(lam), len(lam), _ptr(fid), V,
                                  float(tol), int(maxit), hw, ho, _stream(stream))
    _check(rc, allow_notconv=True)
    return [Path(C.c_void_p(ho[g]), specs[g], rc) for g in range(G)]


def tkm_exact_cv(path: Path, y, foldid, T: int = None, L: int = None, V: int = None, stream=None):
    """The output tables are sized from the path itself; T, L, V, if given, must agree with it."""
    for name, got, want in (("T", T, path.T), ("L", L, path.L), ("V", V, path.V)):
        if got is not None and got != want:
            raise ValueError("tkm_exact_cv: %s = %d but the path was fitted with %s = %d" % (name, got, name, want))
    T, L, V = path.T, path.L, path.V
    y = _dev_vec(y, path.n, "y")
    fid = _fold_vec(foldid, path.n, V)
    cv_loss = np.empty((T, L, V))
    cv_err = np.empty((T, L, V), dtype=np.int64)
    cv_mean = np.empty((T, L))
    best = np.empty(T, dtype=np.int32)
    _check(lib().tkm_exact_cv(path._h, y.data_ptr(), _ptr(fid), _ptr(cv_loss), _ptr(cv_err), _ptr(cv_mean),
                              _ptr(best), _stream(stream)))
    return cv_loss, cv_err, cv_mean, best


def tkm_path_duality_gap(path: Path, y, foldid, stream=None):
    """(primal, gap) per column of a hinge / quantile path: objective of the non-smoothed problem and its
    duality-gap certificate (reading G22)."""
    y = _dev_vec(y, path.n, "y")
    fid = _fold_vec(foldid, path.n, path.V)
    primal, gap = np.empty(path.B), np.empty(path.B)
    _check(lib().tkm_path_duality_gap(path._h, y.data_ptr(), _ptr(fid), _ptr(primal), _ptr(gap), _stream(stream)))
    return primal, gap


def tkm_cv_select(cv_loss, fold_sizes, lambdas, stream=None):
    """Pooled CV mean and selected lambda from a T x L x V fold-loss table (host arrays)."""
    cv_loss = _host(cv_loss, np.float64)
    T, L, V = cv_loss.shape
    fs = _host(fold_sizes, np.float64)
    lam = _host(lambdas, np.float64)
    assert fs.shape == (V,) and lam.shape == (L,)
    cv_mean = np.empty((T, L))
    best = np.empty(T, dtype=np.int32)
    _check(lib().tkm_cv_select(_ptr(cv_loss), _ptr(fs), _ptr(lam), T, L, V, _ptr(cv_mean), _ptr(best),
                               _stream(stream)))
    return cv_mean, best


def tkm_fit_cv_sharded(spec: Spectral, y, loss: int, lambdas, foldid, V: int, tol: float, maxit: int, dist=None,
                       rank=None, world=None, taus=None, stream=None, **fit_kw):
    """Column sharding over GPUs: this rank fits the lambdas `ranks.lambda_slice` gives it
    (interleaved: the iteration count grows as lambda falls) for every fold and variant, runs exact CV on
    its own columns, the ranks exchange the fold-loss tables (kilobytes; the only communication), and every
    rank selects lambda from the full table.  Returns (path of this rank's lambdas, their indices in
    `lambdas`, cv_loss, cv_err, cv_mean, best) with the tables in the full grid's order."""
    from . import ranks
    if rank is None:
        rank = dist.get_rank() if dist is not None and dist.is_initialized() else 0
    if world is None:
        world = dist.get_world_size() if dist is not None and dist.is_initialized() else 1
    lam = _host(lambdas, np.float64)
    mine = ranks.lambda_slice(len(lam), rank, world)
    T = len(taus) if taus is not None and len(taus) else 1
    path = tkm_fit_path(spec, y, loss, lam[mine], foldid, V, tol, maxit, taus=taus, stream=stream, **fit_kw)
    loc_loss, loc_err, _, _ = tkm_exact_cv(path, y, foldid, T, len(mine), V, stream=stream)
    cv_loss = ranks.gather_lambda_tables(loc_loss, len(lam), rank, world, dist)
    cv_err = ranks.gather_lambda_tables(loc_err, len(lam), rank, world, dist)
    fid = _host(foldid, np.int32)
    fsize = np.empty(V)
    _check(lib().tkm_fold_sizes(_ptr(fid), len(fid), V, _ptr(fsize)))
    cv_mean, best = tkm_cv_select(cv_loss, fsize, lam, stream=stream)
    return path, mine, cv_loss, cv_err, cv_mean, best


def tkm_path_coef(path: Path, t: int, l: int, v: int, stream=None):
    import torch
    n = path.spec.n
    out = torch.empty(n, device="cuda", dtype=torch.float64)   # Nystrom: first m entries are used
    b0 = C.c_double()
    _check(lib().tkm_path_coef(path._h, t, l, v, out.data_ptr(), C.byref(b0), _stream(stream)))
    return out, b0.value


def tkm_predict(path: Path, t: int, l: int, X_train, X_new, sigma: float, labels=True, stream=None):
    import torch
    X_train, X_new = _dev_f64(X_train, "X_train"), _dev_f64(X_new, "X_new")
    n_new, p = X_new.shape
    f = torch.empty(n_new, device="cuda", dtype=torch.float64)
    lab = torch.empty(n_new, device="cuda", dtype=torch.int8) if labels else None
    _check(lib().tkm_predict(path._h, t, l, X_train.data_ptr(), X_train.stride(0), X_new.data_ptr(), n_new,
                             X_new.stride(0), p, float(sigma), f.data_ptr(),
                             lab.data_ptr() if lab is not None else None, _stream(stream)))
    return f, lab


PREDICT_NOALLOC_MAX_COEF = 65536


def tkm_predict_noalloc(path: Path, t: int, l: int, X_train, X_new, sigma: float, f_out, label_out=None, stream=None):
    """tkm_predict without any allocation (include/tkm.h): the caller passes the outputs (f_out: n_new FP64 on the
    device, label_out: n_new int8 or None); asynchronous on `stream`."""
    import torch
    X_train, X_new = _dev_f64(X_train, "X_train"), _dev_f64(X_new, "X_new")
    n_new, p = X_new.shape
    if not (f_out.is_cuda and f_out.dtype == torch.float64 and f_out.is_contiguous() and f_out.numel() >= n_new):
        raise ValueError("f_out: contiguous float64 CUDA tensor of n_new elements")
    if label_out is not None and not (label_out.is_cuda and label_out.dtype == torch.int8 and
                                      label_out.is_contiguous() and label_out.numel() >= n_new):
        raise ValueError("label_out: contiguous int8 CUDA tensor of n_new elements")
    _check(lib().tkm_predict_noalloc(path._h, t, l, X_train.data_ptr(), X_train.stride(0), X_new.data_ptr(), n_new,
                                     X_new.stride(0), p, float(sigma), f_out.data_ptr(),
                                     label_out.data_ptr() if label_out is not None else None, _stream(stream)))
    return f_out, label_out


def tkm_train_tune_host(X, y, sigmas, loss, lambdas, foldid, V, tol, maxit, smooth0=1.0, eta=0.125, rounds=4,
                        taus=None, restart=True, check_every=0, warm_tol=0.0,
                        want_alpha=True, tf32_delta=False, stream=None):
    """Whole pipeline from HOST numpy buffers for G bandwidths at once (the `e2e` call of bench.py)."""
    X = _host(X, np.float64)
    y = _host(y, np.float64)
    lam = _host(lambdas, np.float64)
    fid = _host(foldid, np.int32)
    sig = _host(np.atleast_1d(sigmas), np.float64)
    G = len(sig)
    n, p = X.shape
    o, keep = _opts(loss, smooth0, eta, rounds, taus, restart, check_every, warm_tol, False, tf32_delta)
    T, L = max(1, len(keep)), len(lam)
    cv_loss = np.empty((G, T, L, V))
    cv_err = np.empty((G, T, L, V), dtype=np.int64)
    cv_mean = np.empty((G, T, L))
    best = np.empty((G, T), dtype=np.int32)
    alpha = np.empty((G, n)) if want_alpha else None
    b0 = np.zeros(G)
    stage = np.zeros(5, dtype=np.float32)
    rc = lib().tkm_train_tune_host(_ptr(X), n, p, _ptr(y), _ptr(sig), G, loss, C.byref(o), _ptr(lam), L, _ptr(fid),
                                   V, float(tol), int(maxit), _ptr(cv_loss), _ptr(cv_err),
                                   _ptr(cv_mean), _ptr(best), _ptr(alpha) if want_alpha else None, _ptr(b0),
                                   _ptr(stage), _stream(stream))
    _check(rc, allow_notconv=True)
    return dict(cv_loss=cv_loss, cv_err=cv_err, cv_mean=cv_mean, best_l=best, alpha=alpha, beta0=b0,
                stage_ms=stage, status=rc)


def tkm_dgemm_nt(P, Q, stream=None):
    """Dt[N][M] = P[N][K] Q[M][K]^T on the library's DMMA kernel (probe / tests)."""
    import torch
    P, Q = _dev_f64(P, "P"), _dev_f64(Q, "Q")
    N, K = P.shape
    M = Q.shape[0]
    ldd = (M + 1) // 2 * 2
    D = torch.empty((N, ldd), device="cuda", dtype=torch.float64)
    _check(lib().tkm_dgemm_nt(P.data_ptr(), P.stride(0), Q.data_ptr(), Q.stride(0), D.data_ptr(), ldd, N, M, K,
                              _stream(stream)))
    return D[:, :M]


def tkm_gemm_probe(cfg: int, G: int, N: int, M: int, K: int, iters: int = 20, stream=None) -> float:
    """Milliseconds per launch of the library's DMMA GEMM on synthetic operands (roofline calibration)."""
    ms = C.c_float()
    _check(lib().tkm_gemm_probe(cfg, G, N, M, K, iters, C.byref(ms), _stream(stream)))
    return float(ms.value)


def tkm_tf32x3_gemm_nt(P, Q, cfg=-1, iters=0, stream=None):
    """Dt[N][M] = P[N][K] Q[M][K]^T on the 3xTF32 tcgen05 kernel (FP64 in/out, FP32 accumulation).
    Returns D, or (D, ms per launch) when iters > 0."""
    import torch
    P, Q = _dev_f64(P, "P"), _dev_f64(Q, "Q")
    N, K = P.shape
    M = Q.shape[0]
    D = torch.empty((N, M), device="cuda", dtype=torch.float64)
    ms = C.c_float()
    _check(lib().tkm_tf32x3_gemm_nt(P.data_ptr(), P.stride(0), Q.data_ptr(), Q.stride(0), D.data_ptr(), M, N, M, K,
                                    cfg, iters, C.byref(ms) if iters > 0 else None, _stream(stream)))
    return (D, float(ms.value)) if iters > 0 else D


def tkm_cv_decision_values(path: Path, t: int, l: int, foldid, stream=None):
    """Held-out decision value of every training row at (t, lambda_l) from the exact-CV columns."""
    import torch
    fid = _fold_vec(foldid, path.n, path.V)
    f = torch.empty(path.spec.n, device="cuda", dtype=torch.float64)
    _check(lib().tkm_cv_decision_values(path._h, t, l, _ptr(fid), f.data_ptr(), _stream(stream)))
    return f


def tkm_platt_fit(f, y, stream=None):
    """(A, B, iterations) of Platt's sigmoid 1 / (1 + exp(A f + B))."""
    f, y = _dev_f64(f, "f"), _dev_f64(y, "y")
    A, B, it = C.c_double(), C.c_double(), C.c_int32()
    _check(lib().tkm_platt_fit(f.data_ptr(), y.data_ptr(), f.numel(), C.byref(A), C.byref(B), C.byref(it),
                               _stream(stream)))
    return A.value, B.value, it.value


def tkm_platt_proba(f, A: float, B: float, stream=None):
    import torch
    f = _dev_f64(f, "f")
    p = torch.empty_like(f)
    _check(lib().tkm_platt_proba(f.data_ptr(), f.numel(), float(A), float(B), p.data_ptr(), _stream(stream)))
    return p
