"""Oracle of the factorisation-free approximate projection.

TEST INFRASTRUCTURE, NOT THE PRODUCT (only tests/ and bench.py's cpu_baseline leg may import it).  Plain numpy,
complex128; shares nothing with paper_2606_20519_b200/.

The paper's outlook (b): "the corresponding spectral map can be approximated by a composite matrix polynomial
constructed solely from matrix-matrix products, with coefficients optimized to reproduce the eigenvalue-thresholding
operation", citing ref. [81], whose coefficients are NOT in this container.  Reading taken (DESIGN.md
section 4): the composite polynomial is the K-fold composition of the Newton-Schulz cubic g(t) = (3 t - t^3) / 2, the
textbook polynomial iteration for the matrix sign function, applied to X / s with s = ||X||_F (an upper bound of the
spectral radius, so every eigenvalue of X / s lies in [-1, 1] where the iteration converges monotonically to sign):

    S_0 = X / s,      S_{k+1} = (3 S_k - S_k^3) / 2   (k = 0 .. K-1),      P_K = (X + X S_K) / 2.

P_K is the polynomial filter lambda -> lambda (1 + g^K(lambda / s)) / 2 applied to the spectrum of X; it is "parity
unpinned" with respect to the paper's OWN coefficients (they are not available), and pinned as an algorithm by the
scalar recurrence, the exact projection and the error identity in tests/test_oracle_approx.py.
"""
from __future__ import annotations

import numpy as np


def scalar_filter(t: np.ndarray, iterations: int) -> np.ndarray:
    """g^K(t), the K-fold composition of g(t) = (3 t - t^3)/2, on real numbers (the spectrum of X / s)."""
    t = np.array(t, dtype=float)
    for _ in range(iterations):
        t = 0.5 * (3.0 * t - t * t * t)
    return t


def project_approx(X: np.ndarray, iterations: int) -> np.ndarray:
    """P_K(X) as defined above, step by step, with matrix products only."""
    X = np.asarray(X, dtype=complex)
    s = np.linalg.norm(X)                     # Frobenius norm
    if s == 0.0:
        return np.zeros_like(X)
    S = X / s
    for _ in range(iterations):
        T = S @ S
        S = 1.5 * S - 0.5 * (S @ T)
    return 0.5 * (X + X @ S)
