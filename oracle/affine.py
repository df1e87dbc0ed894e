"""Oracle of the affine-projection step of the paper's SCS solver.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may
import this.  Plain numpy in complex128 / float64, written from the paper's definitions, in the paper's notation;
it shares no code with paper_2606_20519_b200/ and imports nothing from it.

What it computes (bipartite scenario, all four local dimensions equal to d, subsystem order A_i, A_o, B_i, B_o,
n = d^4 = d_tot):
  * gell_mann(d):     the orthonormal Hermitian basis {sigma_alpha} of Eq. (A10):
                      identity / sqrt(d); d-1 diagonal elements; (|j><k| + |k><j|)/sqrt 2; -i(|j><k| - |k><j|)/sqrt 2.
  * allowed_indices(d): the multi-indices (alpha, beta, gamma, delta) of Eq. (B14):
                      w_{alpha 0, gamma 0},  w_{i 0, gamma l},  w_{alpha j, k 0}   (Greek: any, Latin: traceless, >= 1),
                      without the all-identity index (its coefficient is fixed by the trace).
                      Order: lexicographic in (alpha, beta, gamma, delta) -- the paper fixes none (DESIGN.md readings).
  * F_mu = sigma_alpha (x) sigma_beta (x) sigma_gamma (x) sigma_delta   (Eq. B10; orthonormal: D4)
  * apply_A(x)  = - sum_mu x_mu F_mu,     apply_AT(Z)_mu = - tr[F_mu Z]      (Eq. D3)
  * affine_project(a_x, a_y):  z_x = (a_x - A^T a_y) / 2,  z_y = a_y + A z_x
Matrices cross this module as dense Hermitian n x n arrays; the svec encoding is oracle.pack / oracle.unpack.

apply_A_explicit / apply_AT_explicit form every F_mu as a dense Kronecker product (the definition written out; small d
only).  apply_A / apply_AT contract over the local basis tensors with numpy.einsum, which is how the paper evaluates
them; tests pin the two against each other and both against (D4), (D5) and Table II.
"""
from __future__ import annotations

import numpy as np


def gell_mann(d: int) -> np.ndarray:
    """(d^2, d, d) complex: sigma_0 .. sigma_{d^2-1} of Eq. (A10), in the order the equation lists them."""
    out = [np.eye(d, dtype=complex) / np.sqrt(d)]
    for l in range(d - 1):                                   # 0 <= l <= d-2
        m = np.zeros((d, d), dtype=complex)
        for j in range(l + 1):
            m[j, j] = 1.0
        m[l + 1, l + 1] = -(l + 1)
        out.append(np.sqrt(1.0 / ((l + 1) * (l + 2))) * m)
    for j in range(d):
        for k in range(j + 1, d):
            m = np.zeros((d, d), dtype=complex)
            m[j, k] = 1.0
            m[k, j] = 1.0
            out.append(m / np.sqrt(2.0))
    for j in range(d):
        for k in range(j + 1, d):
            m = np.zeros((d, d), dtype=complex)
            m[j, k] = -1j
            m[k, j] = 1j
            out.append(m / np.sqrt(2.0))
    return np.array(out)


def allowed_indices(d: int) -> np.ndarray:
    """(m, 4) int array of the allowed multi-indices of Eq. (B14), all-identity excluded, lexicographic order."""
    q = d * d
    idx = []
    for al in range(q):
        for be in range(q):
            for ga in range(q):
                for de in range(q):
                    if al == 0 and be == 0 and ga == 0 and de == 0:
                        continue
                    ok = (be == 0 and de == 0) or (al >= 1 and be == 0 and de >= 1) or (be >= 1 and ga >= 1 and de == 0)
                    if ok:
                        idx.append((al, be, ga, de))
    return np.array(idx, dtype=np.int64)


def n_constraints(d: int) -> int:
    """m = 2 d^6 - 3 d^4 + 2 d^2 - 1 (PAPER.md:729 minus the fixed identity coefficient; column m of Table II)."""
    return 2 * d ** 6 - 3 * d ** 4 + 2 * d ** 2 - 1


def basis_element(sig: np.ndarray, mu) -> np.ndarray:
    al, be, ga, de = (int(t) for t in mu)
    return np.kron(np.kron(sig[al], sig[be]), np.kron(sig[ga], sig[de]))


def apply_A_explicit(d: int, x: np.ndarray) -> np.ndarray:
    sig, idx = gell_mann(d), allowed_indices(d)
    W = np.zeros((d ** 4, d ** 4), dtype=complex)
    for xm, mu in zip(x, idx):
        W -= xm * basis_element(sig, mu)
    return W


def apply_AT_explicit(d: int, Z: np.ndarray) -> np.ndarray:
    sig, idx = gell_mann(d), allowed_indices(d)
    return np.array([-np.trace(basis_element(sig, mu) @ Z).real for mu in idx])


def _coeff_tensor(d: int, x: np.ndarray) -> np.ndarray:
    q = d * d
    w = np.zeros((q, q, q, q))
    idx = allowed_indices(d)
    w[idx[:, 0], idx[:, 1], idx[:, 2], idx[:, 3]] = x
    return w


def apply_A(d: int, x: np.ndarray) -> np.ndarray:
    """A x = - sum_mu x_mu F_mu by contraction over the local bases."""
    sig = gell_mann(d)
    w = _coeff_tensor(d, np.asarray(x, dtype=float))
    # W[(a b c e), (a' b' c' e')] = sum w[al,be,ga,de] sig[al][a,a'] sig[be][b,b'] sig[ga][c,c'] sig[de][e,e']
    t = np.einsum("pqrs,pai,qbj,rck,sel->abceijkl", w, sig, sig, sig, sig, optimize=True)
    return -t.reshape(d ** 4, d ** 4)


def apply_AT(d: int, Z: np.ndarray) -> np.ndarray:
    """(A^T Z)_mu = - tr[F_mu Z] by contraction over the local bases."""
    sig = gell_mann(d)
    z = np.asarray(Z, dtype=complex).reshape((d,) * 8)       # [a b c e, a' b' c' e']
    # tr[F Z] = sum F[(abce),(ijkl)] Z[(ijkl),(abce)]
    t = np.einsum("pai,qbj,rck,sel,ijklabce->pqrs", sig, sig, sig, sig, z, optimize=True)
    idx = allowed_indices(d)
    return -t[idx[:, 0], idx[:, 1], idx[:, 2], idx[:, 3]].real


def affine_project(d: int, a_x: np.ndarray, a_y: np.ndarray):
    """z = M^{-1} a with M = [[1, A^T], [-A, 1]] and A^T A = 1:  z_x = (a_x - A^T a_y)/2,  z_y = a_y + A z_x
    (PAPER.md:1522-1528).  a_y, z_y are Hermitian n x n matrices."""
    z_x = 0.5 * (np.asarray(a_x, dtype=float) - apply_AT(d, a_y))
    z_y = np.asarray(a_y, dtype=complex) + apply_A(d, z_x)
    return z_x, z_y


# ---- the process projector of Eq. (B4), written from the trace-and-replace definition (A1): used ONLY to pin A A^T (D5)
def _trace_and_replace(M: np.ndarray, d: int, subsystems) -> np.ndarray:
    """_X M = 1_X / d_X (x) tr_X M for X a set of the four subsystems (0: A_i, 1: A_o, 2: B_i, 3: B_o), Eq. (A1)."""
    t = M.reshape((d,) * 8)
    for s in subsystems:
        tr = np.trace(t, axis1=s, axis2=4 + s)                         # removes both axes of subsystem s
        eye = np.eye(d) / d
        t = np.einsum("...,ij->...ij", tr, eye)                        # appended as the last two axes
        # move the two new axes back to positions s and 4 + s
        t = np.moveaxis(t, [-2, -1], [s, 4 + s])
    return t.reshape(d ** 4, d ** 4)


def process_projector(M: np.ndarray, d: int) -> np.ndarray:
    """P_proc[M] of Eq. (B4)."""
    T = lambda *s: _trace_and_replace(M, d, s)
    return T(1) + T(3) - T(1, 3) - T(0, 1) - T(2, 3) + T(1, 2, 3) + T(0, 1, 3)
