"""Pins P1, P2, P14 for the oracle: Gram, eigendecomposition, folds."""
import os

import numpy as np
import pytest

import oracle as o
import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_gram_two_point_closed_form():
    # P1: ||x - x'|| = 5 (3-4-5 triangle), sigma = 2.5  =>  k = exp(-25 / 12.5) = exp(-2)
    X = np.array([[0.0, 0.0], [3.0, 4.0]])
    K = o.gram_rbf(X, 2.5)
    assert K[0, 1] == pytest.approx(np.exp(-2.0), rel=1e-15)
    assert K[0, 0] == 1.0 and K[1, 1] == 1.0
    # sigma is a LENGTH (G12): doubling sigma takes the exponent to -1/2
    assert o.gram_rbf(X, 5.0)[0, 1] == pytest.approx(np.exp(-0.5), rel=1e-15)


def test_gram_invariants_and_library_routine():
    w = wl.config0(n=150, p=7, seed=3)
    K = o.gram_rbf(w.X, w.sigmas[0])
    assert np.array_equal(K, K.T)                       # bit-exact symmetry
    assert np.all(np.diag(K) == 1.0)
    assert np.all(K > 0) and np.all(K <= 1.0)
    assert np.linalg.eigvalsh(K).min() >= -w.n * np.finfo(float).eps
    # special case that reduces to a library routine: scipy's squared-Euclidean cdist
    from scipy.spatial.distance import cdist
    ref = np.exp(-cdist(w.X, w.X, "sqeuclidean") / (2 * w.sigmas[0] ** 2))
    assert np.max(np.abs(K - ref)) < 1e-14


def test_gram_cross():
    rng = np.random.default_rng(0)
    A, Bm = rng.standard_normal((9, 4)), rng.standard_normal((5, 4))
    K = o.gram_rbf(A, 1.3, Bm)
    assert K.shape == (9, 5)
    for i in (0, 8):
        for j in (0, 4):
            assert K[i, j] == pytest.approx(np.exp(-np.sum((A[i] - Bm[j]) ** 2) / (2 * 1.3 ** 2)), rel=1e-14)
    with pytest.raises(ValueError):
        o.gram_rbf(A, 0.0)


def test_spectral_invariants(tiny_problem):
    # P2: U^T U = I, U Lam U^T = K, Lam >= 0, u1 = U^T 1
    K, spec = tiny_problem["K"], tiny_problem["spec"]
    n = K.shape[0]
    assert np.max(np.abs(spec.U.T @ spec.U - np.eye(n))) < 1e-12 * n
    assert np.max(np.abs((spec.U * spec.lam) @ spec.U.T - K)) < 1e-12 * n
    assert np.all(spec.lam >= 0)
    assert np.allclose(spec.u1, spec.U.sum(axis=0), atol=1e-13)
    assert abs(spec.u1 @ spec.u1 - n) < 1e-10          # ||U^T 1||^2 = n for orthogonal U


def test_splitmix64_reference_vector():
    # P14: first outputs of SplitMix64 for seed 1234567 (the published reference vector of
    # the generator; stored in tests/golden/splitmix64_seed1234567.txt with its citation).
    want = [int(ln) for ln in open(os.path.join(GOLDEN, "splitmix64_seed1234567.txt"))
            if ln.strip() and not ln.startswith("#")]
    g = o.splitmix64_stream(1234567)
    got = [next(g) for _ in range(len(want))]
    assert got == want and len(want) == 5


@pytest.mark.parametrize("n,V,seed", [(200, 5, 7), (17, 4, 0), (10, 10, 3), (1001, 10, 2**63 + 5)])
def test_folds_invariants(n, V, seed):
    f = o.make_folds(n, V, seed)
    assert f.dtype == np.int32 and f.shape == (n,)
    sizes = np.bincount(f, minlength=V)
    assert sizes.sum() == n and set(sizes) <= {n // V, -(-n // V)}
    assert np.array_equal(f, o.make_folds(n, V, seed))          # same seed => same bytes
    if n > 20:
        assert not np.array_equal(f, o.make_folds(n, V, seed + 1))


def test_folds_tiny_brute_force():
    # n = 4, V = 2: replay Fisher-Yates by hand from the raw stream
    g = o.splitmix64_stream(42)
    r = [next(g) for _ in range(3)]
    pi = [0, 1, 2, 3]
    for i, x in zip((3, 2, 1), r):
        j = x % (i + 1)
        pi[i], pi[j] = pi[j], pi[i]
    want = np.empty(4, dtype=np.int32)
    for i in range(4):
        want[pi[i]] = i % 2
    assert np.array_equal(o.make_folds(4, 2, 42), want)
    with pytest.raises(ValueError):
        o.make_folds(3, 5, 1)
