"""Pins of the approximate-projection oracle (oracle/approx.py, NEXT-4): the matrix iteration against the SCALAR
recurrence on a known spectrum (no matrix product involved), the error identity against the exact projection, its
monotone decay in K, and special cases."""
import numpy as np
import pytest

from oracle import approx
import workloads


def spectral(rng, n, lam):
    g = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    q, r = np.linalg.qr(g)
    q = q * (np.diag(r) / np.abs(np.diag(r)))[None, :]
    X = (q * lam[None, :]) @ q.conj().T
    return 0.5 * (X + X.conj().T), q


@pytest.mark.parametrize("K", [0, 1, 5, 12, 30])
def test_matrix_iteration_is_the_scalar_filter_on_the_spectrum(K):
    rng = np.random.default_rng(3 + K)
    n = 40
    lam = rng.standard_normal(n)
    X, q = spectral(rng, n, lam)
    s = np.linalg.norm(lam)
    want = (q * (0.5 * lam * (1.0 + approx.scalar_filter(lam / s, K)))[None, :]) @ q.conj().T
    got = approx.project_approx(X, K)
    assert np.linalg.norm(got - want) <= 1e-12 * np.linalg.norm(X)


def test_error_identity_and_convergence_to_the_exact_projection():
    rng = np.random.default_rng(11)
    n = 48
    lam = np.concatenate([rng.uniform(0.5, 2.0, 4), rng.normal(0, 1e-2, n - 4)])
    X, q = spectral(rng, n, lam)
    exact = (q * np.maximum(lam, 0)[None, :]) @ q.conj().T
    s = np.linalg.norm(lam)
    prev = np.inf
    for K in (5, 10, 20, 30, 40):
        err = np.linalg.norm(approx.project_approx(X, K) - exact)
        bound = 0.5 * np.linalg.norm(lam * (1.0 - np.abs(approx.scalar_filter(lam / s, K))))   # an identity, not only a bound
        assert abs(err - bound) <= 1e-12 * np.linalg.norm(X)
        assert err <= prev + 1e-14
        prev = err
    assert prev <= 1e-9 * np.linalg.norm(X)


def test_special_cases():
    assert np.all(approx.project_approx(np.zeros((5, 5)), 7) == 0)
    d = np.diag([2.0, -1.0, 0.5, -0.25]).astype(complex)
    p = approx.project_approx(d, 60)
    assert np.allclose(p, np.diag([2.0, 0.0, 0.5, 0.0]), atol=1e-12)
    x = np.eye(6) * 3.0
    assert np.allclose(approx.project_approx(x, 60), x, atol=1e-12)
    assert np.allclose(approx.project_approx(-x, 60), 0, atol=1e-12)
    assert approx.scalar_filter(np.array([1.0, -1.0, 0.0]), 9).tolist() == [1.0, -1.0, 0.0]     # fixed points of g
