"""Pins for the CPU oracle (oracle/hpsd_oracle.c) against what the paper and the
mathematics fix -- never against the oracle itself, never against the CUDA path.

Each test names the passage or identity it checks (SURVEY.md §8(c) pin table).
"""
import os

import numpy as np
import pytest

import workloads
from conftest import rel_err

GOLD = os.path.join(os.path.dirname(__file__), "golden")
EPS = 2.0 ** -52
S2 = np.sqrt(2.0)


def psd_closed_form(b):
    """Q diag(max(lam,0)) Q^H from the GENERATOR's Q and lam: no eigensolver."""
    return (b.Q * np.maximum(b.lam, 0.0)[None, :]) @ b.Q.conj().T


def herm(rng, n, scale=1.0):
    g = (rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))) * scale
    return 0.5 * (g + g.conj().T)


def proj_mat(orc, X):
    n = X.shape[0]
    return orc.unpack(orc.project([n], orc.pack(X)), n)


# ---------------------------------------------------------------- layout (D10)

def test_golden_table3_sizes():
    """n = d^4 for d = 2..8, PAPER.md:1510-1518 (Table III)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "table3_sizes.txt")) if not l.startswith("#")]
    assert [(int(d), int(n)) for d, n in rows] == [(d, d ** 4) for d in range(2, 9)]


def test_golden_vecR_worked_3x3(orc):
    """Hand-worked vec_R of a 3x3 matrix, Eq. (D10) PAPER.md:1222."""
    X = np.array([[2, 1 - 2j, 3 + 1j], [1 + 2j, -1, -4j], [3 - 1j, 4j, 5]], dtype=np.complex128)
    want = np.zeros(9)
    for l in open(os.path.join(GOLD, "vecR_worked_3x3.txt")):
        if l.startswith("#"):
            continue
        i, kind, v = l.split()
        want[int(i)] = float(v) * (S2 if kind == "s" else 1.0)
    got = orc.pack(X)
    assert np.array_equal(got, want)
    assert np.array_equal(orc.unpack(got, 3).real, X.real)
    np.testing.assert_allclose(orc.unpack(got, 3), X, rtol=0, atol=4 * EPS * 5)


@pytest.mark.parametrize("n", [1, 2, 3, 16, 81, 200])
def test_layout_roundtrip_and_inner_product(orc, n):
    """vec_R(X)^T vec_R(Y) = tr[X^H Y] and mat_R(vec_R(X)) = X."""
    rng = np.random.default_rng(n)
    X, Y = herm(rng, n), herm(rng, n)
    sx, sy = orc.pack(X), orc.pack(Y)
    assert sx.shape == (n * n,)
    np.testing.assert_allclose(orc.unpack(sx, n), X, rtol=0, atol=4 * EPS * np.abs(X).max())
    tr = np.trace(X.conj().T @ Y)
    assert abs(tr.imag) <= 1e-12 * (1 + abs(tr))
    assert abs(sx @ sy - tr.real) <= 64 * EPS * n * np.linalg.norm(X) * np.linalg.norm(Y)
    # norm preservation: ||vec_R X||_2 = ||X||_F
    assert abs(np.linalg.norm(sx) - np.linalg.norm(X)) <= 16 * EPS * np.linalg.norm(X)


def test_layout_column_offsets(orc):
    """off(j) = j(2n-j); entry (i,j), i>j: Re at off(j)+1+2(i-j-1), Im one further."""
    n = 7
    for (i, j) in [(0, 0), (3, 3), (6, 6), (1, 0), (6, 0), (4, 2), (6, 5)]:
        X = np.zeros((n, n), dtype=np.complex128)
        if i == j:
            X[i, i] = 3.0
            sv = orc.pack(X)
            assert sv[j * (2 * n - j)] == 3.0 and np.count_nonzero(sv) == 1
        else:
            X[i, j] = 1.0 + 2.0j
            X[j, i] = 1.0 - 2.0j
            sv = orc.pack(X)
            o = j * (2 * n - j) + 1 + 2 * (i - j - 1)
            assert sv[o] == S2 * 1.0 and sv[o + 1] == S2 * 2.0 and np.count_nonzero(sv) == 2
    assert n * (2 * n - n) == n * n


def test_block_offsets_odd_sizes(orc):
    """Block b starts at sum_{c<b} n_c^2: odd n puts later blocks on odd double offsets."""
    rng = np.random.default_rng(5)
    sizes = [3, 5, 2, 1]
    mats = [herm(rng, n) for n in sizes]
    sv = orc.pack_blocks(mats)
    assert sv.shape == (9 + 25 + 4 + 1,)
    back = orc.unpack_blocks(sv, sizes)
    for a, b in zip(back, mats):
        np.testing.assert_allclose(a, b, rtol=0, atol=1e-15 * 10)
    out = orc.project(sizes, sv)
    off = 0
    for n, m in zip(sizes, mats):
        np.testing.assert_array_equal(out[off:off + n * n], orc.project([n], orc.pack(m)))
        off += n * n


def test_conjugate_convention_equivalence(orc):
    """(D10) uses the upper triangle i<j; the library the lower.  Column-major lower
    of X equals row-major upper of conj(X) and P(conj X) = conj P(X), so as a map
    svec -> svec the projection is the same under either convention."""
    rng = np.random.default_rng(77)
    n = 9
    X = herm(rng, n)
    out_lower = orc.project([n], orc.pack(X))
    # reading the same svec numbers as upper-triangle (i<j) data means the matrix conj(X)
    Pc = proj_mat(orc, X.conj())
    np.testing.assert_allclose(orc.unpack(out_lower, n).conj(), Pc, rtol=0, atol=200 * EPS * np.linalg.norm(X))


# ---------------------------------------------------------------- closed forms

@pytest.mark.parametrize("cfg,kw", [(1, {}), (3, dict(n=96)), (3, dict(n=257)),
                                    (5, dict(n=160, n_big=8, n_clusters=4, mult=16))])
def test_closed_form_haar_spectrum(orc, cfg, kw):
    """X = Q diag(lam) Q^H  =>  P = Q diag(max(lam,0)) Q^H, bound 1e-12*n."""
    w = workloads.make(cfg, **kw)
    b = w.blocks[0]
    out = orc.project(w.sizes, orc.pack(b.X))
    ref = orc.pack(psd_closed_form(b))
    assert rel_err(out, ref) <= 200 * EPS * b.n      # far inside 1e-12*n
    assert rel_err(out, ref) <= 1e-12 * b.n


@pytest.mark.slow
def test_closed_form_config3_full(orc):
    """Config 3 at full size n=625 (8 eigenvalues O(1), 617 of size 1e-3)."""
    w = workloads.make(3)
    b = w.blocks[0]
    out = orc.project(w.sizes, orc.pack(b.X), nthreads=orc.max_threads())
    assert rel_err(out, orc.pack(psd_closed_form(b))) <= 200 * EPS * b.n


def test_eigh_residual_and_orthogonality(orc):
    """Eigensolver tolerance: ||XV - VL||_F <= c n eps ||X||_F, ||V^H V - I||_F <= c n eps."""
    w = workloads.make(5, n=128, n_big=8, n_clusters=3, mult=32)
    b = w.blocks[0]
    lam, Z = orc.eigh_svec(orc.pack(b.X), b.n)
    n = b.n
    assert np.linalg.norm(b.X @ Z - Z * lam[None, :]) <= 10 * n * EPS * np.linalg.norm(b.X)
    assert np.linalg.norm(Z.conj().T @ Z - np.eye(n)) <= 10 * n * EPS
    np.testing.assert_allclose(np.sort(lam), np.sort(b.lam), rtol=0, atol=10 * n * EPS * np.abs(b.lam).max())


def test_golden_2x2_worked(orc):
    """Hand-worked 2x2 projections (tests/golden/proj_2x2_worked.txt)."""
    for l in open(os.path.join(GOLD, "proj_2x2_worked.txt")):
        if l.startswith("#") or not l.strip():
            continue
        a, c, br, bi, p00, p11, pr, pi = map(float, l.split())
        X = np.array([[a, br - 1j * bi], [br + 1j * bi, c]])
        P = proj_mat(orc, X)
        want = np.array([[p00, pr - 1j * pi], [pr + 1j * pi, p11]])
        np.testing.assert_allclose(P, want, rtol=0, atol=1e-15 * 8 * max(1.0, np.abs(want).max()))


def test_2x2_analytic_random(orc):
    """lambda_+- = (a+c)/2 +- sqrt(((a-c)/2)^2+|b|^2); mixed signs => P = l+ (X - l- I)/(l+ - l-)."""
    rng = np.random.default_rng(22)
    for _ in range(200):
        a, c = rng.standard_normal(2)
        b = rng.standard_normal() + 1j * rng.standard_normal()
        X = np.array([[a, np.conj(b)], [b, c]])
        r = np.sqrt(((a - c) / 2) ** 2 + abs(b) ** 2)
        lp, lm = (a + c) / 2 + r, (a + c) / 2 - r
        if lm >= 0:
            want = X
        elif lp <= 0:
            want = np.zeros((2, 2))
        else:
            want = lp * (X - lm * np.eye(2)) / (lp - lm)
        np.testing.assert_allclose(proj_mat(orc, X), want, rtol=0, atol=64 * EPS * np.linalg.norm(X))


# ------------------------------------------------ brute force, no eigen-code

def _gauss_jordan_inverse(M):
    n = M.shape[0]
    A = np.concatenate([M.astype(np.complex128), np.eye(n, dtype=np.complex128)], axis=1)
    for c in range(n):
        p = c + int(np.argmax(np.abs(A[c:, c])))
        A[[c, p]] = A[[p, c]]
        A[c] = A[c] / A[c, c]
        for r in range(n):
            if r != c:
                A[r] = A[r] - A[r, c] * A[c]
    return A[:, n:]


def _proj_by_sign_function(X):
    """P = X (I + sign(X))/2 with sign(X) from the Newton iteration S <- (S + S^-1)/2
    (Gauss-Jordan inverses): an eigen-free route (SURVEY §8(c) 'brute force')."""
    S = X.astype(np.complex128)
    for _ in range(200):
        Sn = 0.5 * (S + _gauss_jordan_inverse(S))
        if np.linalg.norm(Sn - S) <= 1e-15 * np.linalg.norm(Sn):
            S = Sn
            break
        S = Sn
    n = X.shape[0]
    P = X @ (np.eye(n) + S) / 2
    return 0.5 * (P + P.conj().T)


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_brute_force_sign_function(orc, n):
    rng = np.random.default_rng(100 + n)
    for _ in range(25):
        X = herm(rng, n)
        want = _proj_by_sign_function(X)
        np.testing.assert_allclose(proj_mat(orc, X), want, rtol=0, atol=1e-11 * np.linalg.norm(X))


# ------------------------------------------------------------------ invariants

def _check_invariants(orc, sizes, sv, c=50):
    """PSD, idempotent, Moreau X = P(X) - P(-X), <P, P-X> = 0,
    P - X = P(-X) is PSD.  Tolerances c n eps ||X||_F."""
    P = orc.project(sizes, sv)
    Pm = orc.project(sizes, -sv)
    PP = orc.project(sizes, P)
    off = 0
    for n in sizes:
        s = slice(off, off + n * n)
        off += n * n
        nx = np.linalg.norm(sv[s])
        tol = c * max(n, 1) * EPS * max(nx, 1e-300)
        assert np.linalg.norm(PP[s] - P[s]) <= tol                      # P(P(X)) = P(X)
        assert np.linalg.norm(sv[s] - (P[s] - Pm[s])) <= tol            # X = P(X) - P(-X)
        assert abs(P[s] @ (P[s] - sv[s])) <= tol * max(nx, 1e-300)      # <P, P - X> = 0
        # PSD as a tolerance test via a shifted Cholesky (no eigensolver involved)
        Pmat = orc.unpack(P[s], n)
        np.linalg.cholesky(Pmat + tol * np.eye(n))
        R = orc.unpack(P[s] - sv[s], n)                                 # P - X >= 0
        np.linalg.cholesky(R + tol * np.eye(n))


def test_invariants_config2_like(orc):
    w = workloads.make(2, n_mats=6, n=81)
    _check_invariants(orc, w.sizes, orc.pack_blocks([b.X for b in w.blocks]))


def test_invariants_config4_like(orc):
    w = workloads.make(4, big=(150, 97), n_small=5, small=36)
    _check_invariants(orc, w.sizes, orc.pack_blocks([b.X for b in w.blocks]))


def test_invariants_small_and_odd(orc):
    rng = np.random.default_rng(9)
    sizes = [1, 2, 5, 16, 33, 0, 64, 65]
    sv = orc.pack_blocks([herm(rng, n) for n in sizes])
    _check_invariants(orc, sizes, sv)


# --------------------------------------------------------------- special cases

def test_special_cases(orc):
    rng = np.random.default_rng(31)
    n = 24
    # diagonal X -> diag(max(x_ii,0)) exactly
    dd = rng.standard_normal(n)
    P = proj_mat(orc, np.diag(dd).astype(np.complex128))
    assert np.array_equal(P, np.diag(np.maximum(dd, 0.0)).astype(np.complex128))
    # PSD X -> X ; NSD X -> 0
    G = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    X = G @ G.conj().T
    np.testing.assert_allclose(proj_mat(orc, X), X, rtol=0, atol=50 * n * EPS * np.linalg.norm(X))
    assert np.linalg.norm(proj_mat(orc, -X)) <= 50 * n * EPS * np.linalg.norm(X)
    # alpha I
    assert np.array_equal(proj_mat(orc, 2.5 * np.eye(n, dtype=np.complex128)), 2.5 * np.eye(n))
    assert np.array_equal(proj_mat(orc, -2.5 * np.eye(n, dtype=np.complex128)), np.zeros((n, n)))
    # zero matrix, n = 1
    assert np.array_equal(proj_mat(orc, np.zeros((n, n), dtype=np.complex128)), np.zeros((n, n)))
    assert orc.project([1], np.array([-3.0]))[0] == 0.0 and orc.project([1], np.array([3.0]))[0] == 3.0
    assert orc.project([], np.zeros(0)).shape == (0,)
    # rank one +- v v^H
    v = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    R = np.outer(v, v.conj())
    np.testing.assert_allclose(proj_mat(orc, R), R, rtol=0, atol=50 * n * EPS * np.linalg.norm(R))
    assert np.linalg.norm(proj_mat(orc, -R)) <= 50 * n * EPS * np.linalg.norm(R)


def test_direct_sum_projects_blockwise(orc):
    rng = np.random.default_rng(32)
    A, B = herm(rng, 7), herm(rng, 12)
    X = np.zeros((19, 19), dtype=np.complex128)
    X[:7, :7], X[7:, 7:] = A, B
    P = proj_mat(orc, X)
    tol = 50 * 19 * EPS * np.linalg.norm(X)
    np.testing.assert_allclose(P[:7, :7], proj_mat(orc, A), rtol=0, atol=tol)
    np.testing.assert_allclose(P[7:, 7:], proj_mat(orc, B), rtol=0, atol=tol)
    assert np.linalg.norm(P[7:, :7]) <= tol


def test_covariances(orc):
    """P(alpha X) = alpha P(X), alpha>0 (power of two: exact); P(U X U^H) = U P(X) U^H
    for permutation and diagonal-phase (+-1, +-i: exactly representable) U."""
    rng = np.random.default_rng(33)
    n = 20
    X = herm(rng, n)
    P = proj_mat(orc, X)
    tol = 50 * n * EPS * np.linalg.norm(X)
    np.testing.assert_allclose(proj_mat(orc, 4.0 * X), 4.0 * P, rtol=0, atol=4 * tol)
    perm = rng.permutation(n)
    np.testing.assert_allclose(proj_mat(orc, X[np.ix_(perm, perm)]), P[np.ix_(perm, perm)], rtol=0, atol=tol)
    ph = np.array([1, -1, 1j, -1j])[rng.integers(0, 4, n)]
    U = np.diag(ph)
    np.testing.assert_allclose(proj_mat(orc, U @ X @ U.conj().T), U @ P @ U.conj().T, rtol=0, atol=tol)


# ------------------------------------------- library as third opinion (not the oracle)

def _numpy_proj(X):
    lam, V = np.linalg.eigh(X)
    return (V * np.maximum(lam, 0.0)[None, :]) @ V.conj().T


@pytest.mark.parametrize("n", [5, 36, 81, 130])
def test_third_opinion_numpy_eigh_and_real_embedding(orc, n):
    """numpy eigh on X, and on the 2n x 2n real-symmetric embedding [[Re,-Im],[Im,Re]]
    whose projection is the embedding of P(X)."""
    rng = np.random.default_rng(n)
    X = herm(rng, n, 1 / np.sqrt(n))
    P = proj_mat(orc, X)
    tol = 100 * n * EPS * np.linalg.norm(X)
    np.testing.assert_allclose(P, _numpy_proj(X), rtol=0, atol=tol)
    E = np.block([[X.real, -X.imag], [X.imag, X.real]])
    PE = _numpy_proj(E)
    np.testing.assert_allclose(P.real, PE[:n, :n].real, rtol=0, atol=tol)
    np.testing.assert_allclose(P.imag, PE[n:, :n].real, rtol=0, atol=tol)


def test_thread_count_does_not_change_result(orc):
    w = workloads.make(3, n=300)
    sv = orc.pack(w.blocks[0].X)
    a = orc.project(w.sizes, sv, nthreads=1)
    b = orc.project(w.sizes, sv, nthreads=4)
    assert np.array_equal(a, b)


def test_admm_step_moreau_pin(orc):
    """Eqs. (D33)-(D34).  Pin by the Moreau decomposition:
    with x = u~ - v, u = P(x) and v_new = u - x = P(x) - x = P(-x), so u >= 0, v_new >= 0 (the PSD cone is
    self-dual), <u, v_new> = 0 and u - v_new = x; and for a closed-form input the values are known."""
    rng = np.random.default_rng(77)
    b = workloads.from_spectrum(rng, np.array([2.0, -1.0, 0.5, -0.25, 3.0, -4.0]))
    n = b.n
    x = orc.pack(b.X)
    v = orc.pack(herm(rng, n))
    ut = x + v
    u, vn = orc.admm_step([n], ut, v)
    want_u = orc.pack((b.Q * np.maximum(b.lam, 0)[None, :]) @ b.Q.conj().T)
    want_v = orc.pack((b.Q * np.maximum(-b.lam, 0)[None, :]) @ b.Q.conj().T)
    assert rel_err(u, want_u) <= 1e-13 and rel_err(vn, want_v) <= 1e-13
    assert abs(u @ vn) <= 1e-13 * np.linalg.norm(u) * np.linalg.norm(vn)
    np.testing.assert_allclose(u - vn, ut - v, rtol=0, atol=1e-13 * np.linalg.norm(x))
