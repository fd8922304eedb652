"""tkm_predict_noalloc (include/tkm.h): the serving call that allocates nothing -- its coefficient scratch is a
static device array -- against the existing tkm_predict on the same fitted column, two calls in a row.  The two entry
points run the same two kernels on the same inputs, so the outputs must be identical; the test states the parity
tolerance the other predict tests use (1e-8 absolute on decision values) and checks bit-equality on top.
Collected last on purpose (file name): the suite runs with `pytest -x`."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


def _fit(tkm, torch, n, seed):
    w = wl.config0(n=n, p=7, L=3, V=3, seed=seed)
    sigma = float(w.sigmas[0])
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X, y = torch.from_numpy(w.X).cuda(), torch.from_numpy(w.y).cuda()
    spec = tkm.tkm_spectral_setup(tkm.tkm_gram(X, sigma))
    path = tkm.tkm_fit_path(spec, y, w.loss, w.lambdas, foldid, w.V, 1e-10, 100000, rounds=w.rounds)
    return w, sigma, X, spec, path


def test_predict_noalloc_matches_predict_on_two_calls_in_a_row():
    import torch
    import paper_2606_06742_b200 as tkm
    tkm.lib()
    torch.cuda.set_device(0)
    # two different fits and two different lambda columns: the second call finds the first call's coefficients in the
    # shared static array (a longer vector than its own) and must not be affected by them
    wa, sa, Xa, spec_a, path_a = _fit(tkm, torch, 333, 5)
    wb, sb, Xb, spec_b, path_b = _fit(tkm, torch, 150, 6)
    cases = [(wa, sa, Xa, path_a, 0, 203), (wb, sb, Xb, path_b, 2, 77), (wa, sa, Xa, path_a, 1, 9)]
    refs = []
    for (w, sigma, X, path, l, n_new) in cases:
        Xn = torch.from_numpy(wl.new_points(w, n_new)).cuda()
        f_ref, lab_ref = tkm.tkm_predict(path, 0, l, X, Xn, sigma)
        refs.append((Xn, f_ref.cpu().numpy(), lab_ref.cpu().numpy()))
    torch.cuda.synchronize()
    outs = []
    for (w, sigma, X, path, l, n_new), (Xn, _, _) in zip(cases, refs):   # back to back on one stream, no sync between
        f = torch.full((n_new,), float("nan"), device="cuda", dtype=torch.float64)
        lab = torch.zeros(n_new, device="cuda", dtype=torch.int8)
        tkm.tkm_predict_noalloc(path, 0, l, X, Xn, sigma, f, lab)
        outs.append((f, lab))
    torch.cuda.synchronize()
    for (f, lab), (_, f_ref, lab_ref) in zip(outs, refs):
        fg = f.cpu().numpy()
        assert np.all(np.isfinite(fg))
        assert np.max(np.abs(fg - f_ref)) <= 1e-8          # the tolerance of the predict parity tests
        assert np.array_equal(fg, f_ref)                    # same kernels, same inputs: the same bits
        assert np.array_equal(lab.cpu().numpy(), lab_ref)
    # without labels
    (w, sigma, X, path, l, n_new), (Xn, f_ref, _) = cases[0], refs[0]
    f = torch.empty(n_new, device="cuda", dtype=torch.float64)
    tkm.tkm_predict_noalloc(path, 0, l, X, Xn, sigma, f, None)
    torch.cuda.synchronize()
    assert np.array_equal(f.cpu().numpy(), f_ref)
    for h in (path_a, path_b, spec_a, spec_b):
        h.close()


def test_predict_noalloc_allocates_nothing():
    """No device allocation between two calls: neither the driver's free memory nor the library pool moves."""
    import torch
    import paper_2606_06742_b200 as tkm
    tkm.lib()
    torch.cuda.set_device(0)
    w, sigma, X, spec, path = _fit(tkm, torch, 200, 8)
    Xn = torch.from_numpy(wl.new_points(w, 64)).cuda()
    f = torch.empty(64, device="cuda", dtype=torch.float64)
    tkm.tkm_predict_noalloc(path, 0, 1, X, Xn, sigma, f)      # first call on this device: the symbol lookup
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        tkm.tkm_predict_noalloc(path, 0, 1, X, Xn, sigma, f)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    path.close()
    spec.close()


def test_predict_noalloc_validates_arguments():
    """Bad (t, l) and sigma come back as errors.  The size limit itself (more than 65536 coefficients -> TKM_EINVAL
    naming TKM_PREDICT_NOALLOC_MAX_COEF) needs a fit with n > 65536 rows of a full kernel or as many Nystrom
    landmarks, which no test can afford; the constant is pinned against the header in tests/test_abi_cpu.py."""
    import torch
    import paper_2606_06742_b200 as tkm
    tkm.lib()
    torch.cuda.set_device(0)
    w, sigma, X, spec, path = _fit(tkm, torch, 120, 9)
    Xn = torch.from_numpy(wl.new_points(w, 5)).cuda()
    f = torch.empty(5, device="cuda", dtype=torch.float64)
    with pytest.raises(tkm.TkmError):
        tkm.tkm_predict_noalloc(path, 0, 99, X, Xn, sigma, f)
    with pytest.raises(tkm.TkmError):
        tkm.tkm_predict_noalloc(path, 0, 0, X, Xn, -1.0, f)
    with pytest.raises(ValueError):
        tkm.tkm_predict_noalloc(path, 0, 0, X, Xn, sigma, f[:3])
    path.close()
    spec.close()
