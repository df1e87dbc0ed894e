"""Pins of the affine-projection oracle (oracle/affine.py) against what the paper and
the mathematics fix, none of them through the oracle's own contraction code:
  * the local basis of Eq. (A10): orthonormal, Hermitian, sigma_0 = 1/sqrt d, the rest traceless (A6)-(A7);
  * the number of allowed multi-indices: column m of Table II and the closed form (B14);
  * A^T A = 1 (D4), A A^T y = P_proc(y) - tr[y]/d_tot 1 (D5) with P_proc written from the trace-and-replace maps
    of Eq. (B4) -- an independent route (partial traces, no basis);
  * the definition written out: dense Kronecker products F_mu for d = 2, 3 against the einsum contraction;
  * the closed form of the affine projection: M z = a with M = [[1, A^T], [-A, 1]] solved densely for d = 2.
"""
import numpy as np
import pytest

from oracle import affine

TABLE_II_M = {2: 87, 3: 1232, 4: 7455, 5: 29424, 6: 89495, 7: 228192, 8: 512127}


def herm(rng, n):
    g = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    return 0.5 * (g + g.conj().T)


@pytest.mark.parametrize("d", [2, 3, 4, 5])
def test_gell_mann_basis_is_orthonormal_hermitian(d):
    s = affine.gell_mann(d)
    assert s.shape == (d * d, d, d)
    assert np.allclose(s, s.conj().transpose(0, 2, 1))
    gram = np.einsum("aij,bji->ab", s, s)
    assert np.allclose(gram, np.eye(d * d), atol=1e-14)
    assert np.allclose(s[0], np.eye(d) / np.sqrt(d))
    assert np.allclose(np.trace(s[1:], axis1=1, axis2=2), 0.0, atol=1e-15)


def test_gell_mann_d2_is_pauli_over_sqrt2():
    s = affine.gell_mann(2)
    r = 1 / np.sqrt(2)
    assert np.allclose(s[1], r * np.array([[1, 0], [0, -1]]))
    assert np.allclose(s[2], r * np.array([[0, 1], [1, 0]]))
    assert np.allclose(s[3], r * np.array([[0, -1j], [1j, 0]]))


@pytest.mark.parametrize("d", sorted(TABLE_II_M))
def test_number_of_constraints_matches_table_ii(d):
    assert affine.n_constraints(d) == TABLE_II_M[d]
    if d <= 5:
        idx = affine.allowed_indices(d)
        assert len(idx) == TABLE_II_M[d]
        assert len({tuple(r) for r in idx}) == len(idx)
        q = d * d
        # (B14): the three families, counted: d^4 - 1 + 2 d^2 (d^2 - 1)^2
        assert len(idx) == q * q - 1 + 2 * q * (q - 1) ** 2


@pytest.mark.parametrize("d", [2, 3])
def test_einsum_contraction_equals_the_definition(d):
    rng = np.random.default_rng(40 + d)
    m = affine.n_constraints(d)
    x = rng.standard_normal(m)
    assert np.allclose(affine.apply_A(d, x), affine.apply_A_explicit(d, x), atol=1e-13)
    Z = herm(rng, d ** 4)
    assert np.allclose(affine.apply_AT(d, Z), affine.apply_AT_explicit(d, Z), atol=1e-13)


def test_basis_elements_are_orthonormal_d2():
    sig, idx = affine.gell_mann(2), affine.allowed_indices(2)
    F = np.array([affine.basis_element(sig, mu).ravel() for mu in idx])
    assert np.allclose(F.conj() @ F.T, np.eye(len(idx)), atol=1e-13)          # tr[F_mu F_nu] = delta (D4)


@pytest.mark.parametrize("d", [2, 3, 4])
def test_AT_A_is_identity(d):
    rng = np.random.default_rng(50 + d)
    x = rng.standard_normal(affine.n_constraints(d))
    W = affine.apply_A(d, x)
    assert np.allclose(W, W.conj().T)
    assert abs(np.trace(W)) < 1e-12                                            # traceless subspace
    assert np.allclose(affine.apply_AT(d, W), x, atol=1e-12)                   # (D4)


@pytest.mark.parametrize("d", [2, 3, 4])
def test_A_AT_is_the_traceless_process_projector(d):
    rng = np.random.default_rng(60 + d)
    n = d ** 4
    Y = herm(rng, n)
    lhs = affine.apply_A(d, affine.apply_AT(d, Y))
    rhs = affine.process_projector(Y, d) - np.trace(Y).real / n * np.eye(n)    # (D5), d_tot = n (garbled subscript)
    assert np.allclose(lhs, rhs, atol=1e-12)
    # P_proc is a projector and A x lies in its range
    P = affine.process_projector(Y, d)
    assert np.allclose(affine.process_projector(P, d), P, atol=1e-12)
    W = affine.apply_A(d, rng.standard_normal(affine.n_constraints(d)))
    assert np.allclose(affine.process_projector(W, d), W, atol=1e-12)


def test_affine_projection_solves_M_z_equals_a_d2():
    """z = M^{-1} a with M = [[1, A^T], [-A, 1]] (D25), solved as a dense real linear system in the vec_R encoding
    (inner-product preserving) for d = 2."""
    import oracle
    d, n = 2, 16
    m = affine.n_constraints(d)
    rng = np.random.default_rng(7)
    # dense real A (n^2 x m) column by column through the definition
    A = np.zeros((n * n, m))
    for k in range(m):
        e = np.zeros(m); e[k] = 1.0
        A[:, k] = oracle.pack(affine.apply_A_explicit(d, e))
    assert np.allclose(A.T @ A, np.eye(m), atol=1e-12)
    M = np.block([[np.eye(m), A.T], [-A, np.eye(n * n)]])
    a_x, a_Y = rng.standard_normal(m), herm(rng, n)
    z = np.linalg.solve(M, np.concatenate([a_x, oracle.pack(a_Y)]))
    z_x, z_Y = affine.affine_project(d, a_x, a_Y)
    assert np.allclose(z[:m], z_x, atol=1e-12)
    assert np.allclose(z[m:], oracle.pack(z_Y), atol=1e-12)
