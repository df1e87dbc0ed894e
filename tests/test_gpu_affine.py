"""GPU parity of the affine-projection step (include/hpsd.h hpsd_affine_*) against the
oracle (oracle/affine.py), through the C ABI: A x, A^T y and z = M^{-1} a element by element for d = 2 .. 5, and the
paper's identities A^T A = 1 (D4) and A A^T y in the traceless process subspace (D5) at d = 6 where the oracle's
einsum takes long.  Tolerance: 1e-12 * n relative 2-norm, as for the projection (same arithmetic type, O(d) terms
per output)."""
import numpy as np
import pytest

from conftest import rel_err

pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def hp():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_20519_b200 as lib
    lib.load_library()
    return lib


def herm(rng, n):
    g = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    return 0.5 * (g + g.conj().T)


@pytest.mark.parametrize("d", [2, 3, 4, 5])
def test_affine_against_oracle(orc, hp, d):
    import torch
    from oracle import affine
    rng = np.random.default_rng(800 + d)
    n = d ** 4
    af = hp.Affine(d)
    try:
        assert (af.n, af.m) == (n, affine.n_constraints(d))
        x = rng.standard_normal(af.m)
        Y = herm(rng, n)
        sv = orc.pack(Y)
        # A x
        got = af.apply_A(torch.from_numpy(x).cuda()).cpu().numpy()
        assert rel_err(got, orc.pack(affine.apply_A(d, x))) <= TOL * n
        # A^T y
        got = af.apply_AT(torch.from_numpy(sv).cuda()).cpu().numpy()
        assert rel_err(got, affine.apply_AT(d, Y)) <= TOL * n
        # z = M^{-1} a, out of place and in place
        zx_w, zy_w = affine.affine_project(d, x, Y)
        tx, ty = torch.from_numpy(x).cuda(), torch.from_numpy(sv).cuda()
        zx, zy = torch.empty_like(tx), torch.empty_like(ty)
        af.project_(tx, ty, zx, zy)
        torch.cuda.synchronize()
        assert rel_err(zx.cpu().numpy(), zx_w) <= TOL * n
        assert rel_err(zy.cpu().numpy(), orc.pack(zy_w)) <= TOL * n
        af.project_(tx, ty, tx, ty)
        torch.cuda.synchronize()
        assert np.array_equal(tx.cpu().numpy(), zx.cpu().numpy())
        assert np.array_equal(ty.cpu().numpy(), zy.cpu().numpy())
    finally:
        af.destroy()


@pytest.mark.parametrize("d", [6])
def test_affine_identities_at_larger_d(orc, hp, d):
    """(D4) A^T A x = x;  M z = a reproduced: z_x + A^T z_y = a_x and z_y - A z_x = a_y (D25), on the GPU output alone."""
    import torch
    rng = np.random.default_rng(820 + d)
    n = d ** 4
    af = hp.Affine(d)
    try:
        x = torch.from_numpy(rng.standard_normal(af.m)).cuda()
        assert rel_err(af.apply_AT(af.apply_A(x)).cpu().numpy(), x.cpu().numpy()) <= TOL * n
        a_x = torch.from_numpy(rng.standard_normal(af.m)).cuda()
        a_y = torch.from_numpy(orc.pack(herm(rng, n))).cuda()
        z_x, z_y = af.project_(a_x, a_y, torch.empty_like(a_x), torch.empty_like(a_y))
        r1 = z_x + af.apply_AT(z_y) - a_x
        r2 = z_y - af.apply_A(z_x) - a_y
        assert float(r1.norm() / a_x.norm()) <= TOL * n
        assert float(r2.norm() / a_y.norm()) <= TOL * n
        # vec_R(A x) is traceless and z_y - a_y lies in the range of A: A A^T (A x) = A x  (D5)
        w = af.apply_A(x)
        assert rel_err(af.apply_A(af.apply_AT(w)).cpu().numpy(), w.cpu().numpy()) <= TOL * n
    finally:
        af.destroy()


# ------------------------------------------------------------------ NEXT-4: approximate projection

@pytest.mark.parametrize("n,K", [(2, 10), (40, 0), (40, 12), (100, 30), (257, 25), (625, 30)])
def test_approximate_projection_against_oracle(orc, hp, n, K):
    """hpsd_project_approx against oracle/approx.py (same K, same polynomial) to 1e-12 n, against the exact projection
    within the error identity 1/2 ||lam (1 - |g^K(lam/s)|)||, and the in-place call."""
    import torch
    from oracle import approx
    rng = np.random.default_rng(870 + n)
    lam = np.concatenate([rng.uniform(0.5, 2.0, min(4, n)), rng.normal(0, 1e-2, max(n - 4, 0))])
    g = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    q, _ = np.linalg.qr(g)
    X = (q * lam[None, :]) @ q.conj().T
    X = 0.5 * (X + X.conj().T)
    sv = orc.pack(X)
    t = torch.from_numpy(sv).cuda()
    got = hp.project_approx(t, n, K).cpu().numpy()
    want = orc.pack(approx.project_approx(X, K))
    assert rel_err(got, want, denom=np.linalg.norm(sv)) <= TOL * n
    exact = orc.pack((q * np.maximum(lam, 0)[None, :]) @ q.conj().T)
    s = np.linalg.norm(sv)
    bound = 0.5 * np.linalg.norm(lam * (1.0 - np.abs(approx.scalar_filter(lam / s, K))))
    assert abs(np.linalg.norm(got - exact) - bound) <= 10 * TOL * n * s
    import ctypes
    rc = hp.load_library().hpsd_project_approx(n, t.data_ptr(), t.data_ptr(), K, None)
    torch.cuda.synchronize()
    assert rc == 0 and np.array_equal(t.cpu().numpy(), got)
