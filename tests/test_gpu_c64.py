"""complex64 storage (complex64 column of Table III):
hpsd_project_c64, hpsd_admm_step_c64, hpsd_plan_*_c64, hpsd_svec_convert through the C ABI.

Oracle: the same FP64 oracle, applied to the FP32 input widened exactly to FP64 (what a complex64 caller holds).
Tolerance, derived from the arithmetic: the library computes the FP64 projection of the widened input
(error <= 1e-12 n, the FP64 parity bound) and rounds every entry to the nearest float (relative error <= 2^-24 per entry,
hence <= 2^-24 in the Frobenius norm), so  ||got - want|| / ||want|| <= 2^-24 + 1e-12 n.  A complex64 eigensolver would be
allowed n 2^-24.  Because the arithmetic IS the FP64 path, the c64 result must also equal, bit for bit, the FP64 entry point's
result on the widened input rounded to float: that pins the load/store conversions on every route."""
import numpy as np
import pytest

from conftest import rel_err

pytestmark = pytest.mark.gpu
EPS32 = 2.0 ** -24
TOL64 = 1e-12


@pytest.fixture(scope="module")
def hp():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_20519_b200 as lib
    lib.load_library()
    return lib


def herm(rng, n, scale=1.0):
    g = (rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))) * scale
    return 0.5 * (g + g.conj().T)


def svec32(orc, rng, sizes):
    """svec of random Hermitian blocks with an O(1) spectrum, rounded to float32 (the caller's storage)."""
    return np.concatenate([orc.pack(herm(rng, n, 1.0 / np.sqrt(max(n, 1)))) for n in sizes]).astype(np.float32)


def check_blocks(got32, want64, sizes, x64):
    off = 0
    for n in sizes:
        sl = slice(off, off + n * n)
        nw, ni = np.linalg.norm(want64[sl]), np.linalg.norm(x64[sl])
        denom = nw if nw > 1e3 * n * 2.2e-16 * ni else max(ni, 1e-300)
        err = rel_err(got32[sl].astype(np.float64), want64[sl], denom=denom)
        assert err <= 1.01 * EPS32 + TOL64 * n, (n, err)
        off += n * n


# every route: scalar, Jacobi, batched D&C medium, in-CTA QL medium, cluster kernel, panel kernel
ROUTES = [[1, 16, 36, 81, 81, 100, 1, 150], [625], [700]]


@pytest.mark.parametrize("sizes", ROUTES, ids=["small_medium_mix", "cluster_625", "panel_700"])
def test_c64_projection_against_oracle_and_fp64_path(orc, hp, sizes):
    import torch
    rng = np.random.default_rng(6400 + sizes[-1])
    sv32 = svec32(orc, rng, sizes)
    x64 = sv32.astype(np.float64)
    want = orc.project(sizes, x64, nthreads=orc.max_threads())
    t_in = torch.from_numpy(sv32).cuda()
    got_t = hp.project(sizes, t_in)
    torch.cuda.synchronize()
    assert got_t.dtype == torch.float32
    got = got_t.cpu().numpy()
    check_blocks(got, want, sizes, x64)
    ref = hp.project(sizes, torch.from_numpy(x64).cuda()).cpu().numpy()
    assert np.array_equal(got, ref.astype(np.float32))        # same arithmetic, only the storage differs
    # in place
    hp.project_(sizes, t_in, t_in)
    torch.cuda.synchronize()
    assert np.array_equal(t_in.cpu().numpy(), got)


def test_c64_two_stage_route(orc, hp):
    import torch
    rng = np.random.default_rng(6411)
    sizes = [200]
    sv32 = svec32(orc, rng, sizes)
    x64 = sv32.astype(np.float64)
    want = orc.project(sizes, x64, nthreads=orc.max_threads())
    hp.set_option("two_stage", 1)
    try:
        got = hp.project(sizes, torch.from_numpy(sv32).cuda()).cpu().numpy()
    finally:
        hp.set_option("two_stage", 0)
    check_blocks(got, want, sizes, x64)


def test_c64_admm_step(orc, hp):
    """Eqs. (D33)-(D34) on complex64 storage: the difference is formed in FP64 from the widened floats, u and the new v are
    rounded once."""
    import torch
    rng = np.random.default_rng(6420)
    sizes = [1, 24, 81, 150, 36, 300]
    ut, v = svec32(orc, rng, sizes), svec32(orc, rng, sizes)
    ut64, v64 = ut.astype(np.float64), v.astype(np.float64)
    want_u, want_v = orc.admm_step(sizes, ut64, v64, nthreads=orc.max_threads())
    t_ut, t_v = torch.from_numpy(ut).cuda(), torch.from_numpy(v.copy()).cuda()
    t_u = torch.empty_like(t_ut)
    hp.admm_step_(sizes, t_ut, t_v, t_u)
    torch.cuda.synchronize()
    check_blocks(t_u.cpu().numpy(), want_u, sizes, ut64 - v64)
    check_blocks(t_v.cpu().numpy(), want_v, sizes, ut64 - v64)
    # against the FP64 entry point on the widened inputs
    d_ut, d_v = torch.from_numpy(ut64).cuda(), torch.from_numpy(v64.copy()).cuda()
    d_u = torch.empty_like(d_ut)
    hp.admm_step_(sizes, d_ut, d_v, d_u)
    torch.cuda.synchronize()
    assert np.array_equal(t_u.cpu().numpy(), d_u.cpu().numpy().astype(np.float32))
    assert np.array_equal(t_v.cpu().numpy(), d_v.cpu().numpy().astype(np.float32))


def test_c64_plan_and_the_single_to_double_switch(orc, hp):
    """One plan serves both storage types (first iterations in single precision, then double): calls alternate,
    replayed graphs are keyed by the storage type, the iterate is widened by hpsd_svec_convert."""
    import torch
    rng = np.random.default_rng(6430)
    sizes = [81, 130, 16]
    sv32 = svec32(orc, rng, sizes)
    t32 = torch.from_numpy(sv32).cuda()
    t64 = hp.svec_convert(t32, torch.float64)
    assert t64.dtype == torch.float64 and np.array_equal(t64.cpu().numpy(), sv32.astype(np.float64))
    back = hp.svec_convert(t64, torch.float32)
    assert np.array_equal(back.cpu().numpy(), sv32)
    plan = hp.Plan(sizes)
    try:
        o32, o64 = torch.empty_like(t32), torch.empty_like(t64)
        first32 = first64 = None
        for it in range(4):                      # plain launches, capture, replays: both kinds interleaved
            plan.project_(t32, o32)
            plan.project_(t64, o64)
            torch.cuda.synchronize()
            if it == 0:
                first32, first64 = o32.cpu().numpy().copy(), o64.cpu().numpy().copy()
            assert np.array_equal(o32.cpu().numpy(), first32) and np.array_equal(o64.cpu().numpy(), first64)
        assert plan.info() == [0, 0, 0]
        assert np.array_equal(first32, first64.astype(np.float32))
        want = orc.project(sizes, sv32.astype(np.float64))
        check_blocks(first32, want, sizes, sv32.astype(np.float64))
        # a short mixed-precision loop: K steps on complex64 storage, widen, continue in double; the fixed point of
        # x <- P(x) is reached after one step, so the widened continuation must reproduce P of the widened iterate
        x32 = t32.clone()
        for _ in range(3):
            plan.project_(x32, x32)
        x64 = hp.svec_convert(x32, torch.float64)
        y64 = plan.project_(x64, torch.empty_like(x64))
        torch.cuda.synchronize()
        want2 = orc.project(sizes, x64.cpu().numpy())
        off = 0
        for n in sizes:
            sl = slice(off, off + n * n)
            assert rel_err(y64.cpu().numpy()[sl], want2[sl]) <= TOL64 * n
            off += n * n
    finally:
        plan.destroy()


def test_c64_non_finite_block(orc, hp):
    import torch
    rng = np.random.default_rng(6440)
    sizes = [40, 130, 20]
    sv32 = svec32(orc, rng, sizes)
    sv32[40 * 40 + 77] = np.inf
    plan = hp.Plan(sizes)
    try:
        t = torch.from_numpy(sv32).cuda()
        out = plan.project_(t, torch.empty_like(t))
        torch.cuda.synchronize()
        assert plan.info() == [0, 2, 0]
        got = out.cpu().numpy()
        assert np.all(np.isnan(got[1600:1600 + 130 * 130]))
        assert np.all(np.isfinite(got[:1600])) and np.all(np.isfinite(got[1600 + 130 * 130:]))
    finally:
        plan.destroy()


def test_c64_rejects_mixed_dtypes(hp):
    import torch
    a = torch.zeros(16, dtype=torch.float32, device="cuda")
    b = torch.zeros(16, dtype=torch.float64, device="cuda")
    with pytest.raises(hp.HpsdError):
        hp.project_([4], a, b)
