"""GPU parity: the CUDA path (through the C ABI, include/hpsd.h) against the CPU oracle on the
same seeded inputs, element by element, plus the projection invariants at sizes where the oracle
takes minutes.  Bar (BASELINE.json north_star): relative Frobenius error <= 1e-12 * n, measured on
the svec vectors (= Frobenius on the matrices); if ||oracle|| = 0 the input norm
is the denominator.  Eigenvectors are never compared (not unique); P(X) is.
"""
import os

import numpy as np
import pytest

import workloads
from conftest import rel_err

pytestmark = pytest.mark.gpu

TOL = 1e-12          # times n
EPS = 2.0 ** -52


@pytest.fixture(scope="module")
def hp():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_20519_b200 as lib
    lib.load_library()          # raises if libhpsd.so is missing: no fallback
    return lib


def _record(what, errs):
    """Append observed parity errors to gpurun_out/parity_observed.txt (a run log, not an expected value)."""
    try:
        os.makedirs("gpurun_out", exist_ok=True)
        with open("gpurun_out/parity_observed.txt", "a") as f:
            f.write(what + ": " + ", ".join(f"n={k} rel_err={v:.3e}" for k, v in errs.items()) + "\n")
    except OSError:
        pass


def check_oracle_samples(cfg, got):
    """Full-size comparison with the ORACLE on sampled outputs (tests/golden/oracle_samples_cfg*.npz, written by
    tests/golden/make_oracle_samples.py, which calls only oracle/): every diagonal entry and every 4099th svec entry
    of the oracle's projection of the whole config, plus the norm of its output."""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"oracle_samples_cfg{cfg}.npz")
    g = np.load(path)
    idx, val = g["idx"], g["val"]
    err = float(np.linalg.norm(got[idx] - val) / np.linalg.norm(val))
    nrm = abs(float(np.linalg.norm(got)) - float(g["norm"])) / float(g["norm"])
    return err, nrm


def force_large(hp, on):
    """Route every block through S1..S8 of the multi-kernel path (on) or restore the defaults (off)."""
    hp.set_option("jacobi_max_n", 1 if on else 32)
    hp.set_option("medium_max_n", 0 if on else 116)


def gpu_project(hp, sizes, sv, **kw):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(sv)).cuda()
    out = hp.project(sizes, t, **kw)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def herm(rng, n, scale=1.0):
    g = (rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))) * scale
    return 0.5 * (g + g.conj().T)


def pack_all(orc, mats):
    return np.concatenate([orc.pack(m) for m in mats]) if mats else np.zeros(0)


def parity_err(got, want, sv_in, n):
    """||got - want|| / ||want||; when the oracle's output is zero or pure rounding noise of a
    negative-semidefinite input (||want|| <= 1e3 n eps ||in||) the input norm is the denominator
    (SURVEY.md §8(c) reading)."""
    nw, ni = np.linalg.norm(want), np.linalg.norm(sv_in)
    denom = nw if nw > 1e3 * max(n, 1) * EPS * ni else max(ni, 1e-300)
    return rel_err(got, want, denom=denom)


def check_vs_oracle(orc, hp, sizes, sv, nthreads=1):
    got = gpu_project(hp, sizes, sv)
    want = orc.project(sizes, sv, nthreads=nthreads)
    off = 0
    for n in sizes:
        a, b = got[off:off + n * n], want[off:off + n * n]
        err = parity_err(a, b, sv[off:off + n * n], n)
        assert err <= TOL * max(n, 1), (n, off, err)
        off += n * n
    return got, want


def _cholesky_ok(M):
    try:
        np.linalg.cholesky(M)
        return True
    except np.linalg.LinAlgError:
        return False


def check_invariants(orc, hp, sizes, sv, out):
    """Projection invariants on the GPU output.  The KKT triple of the projection onto a
    self-dual cone (Moreau) is a COMPLETE certificate of P = Pi(X):
        P >= 0,   P - X >= 0,   <P, P - X> = 0.
    Both semidefiniteness tests are host-side Cholesky factorisations (numpy/LAPACK) of P + tol I and
    (P - X) + tol I, i.e. independent of the library under test; the inner product is an svec dot product
    (PAPER.md:1224-1226).  Idempotence and X = P(X) - P(-X) go through the library again."""
    n = max(sizes)
    nx = np.linalg.norm(sv)
    p2 = gpu_project(hp, sizes, out)
    assert np.linalg.norm(p2 - out) <= TOL * n * nx
    pm = gpu_project(hp, sizes, -sv)
    assert np.linalg.norm(out - pm - sv) <= TOL * n * nx
    assert abs(out @ (out - sv)) <= TOL * n * nx * nx
    off = 0
    for nb in sizes:
        if nb >= 1:
            seg_x, seg_p = sv[off:off + nb * nb], out[off:off + nb * nb]
            tol = TOL * nb * max(np.linalg.norm(seg_x), 1e-300)
            P = orc.unpack(seg_p, nb)
            assert _cholesky_ok(P + tol * np.eye(nb)), ("P not PSD", nb, off)
            assert _cholesky_ok(orc.unpack(seg_p - seg_x, nb) + tol * np.eye(nb)), ("P - X not PSD", nb, off)
            assert abs(seg_p @ (seg_p - seg_x)) <= TOL * nb * max(np.linalg.norm(seg_x), 1e-300) ** 2
        off += nb * nb


# ------------------------------------------------------------------ layout kernels (S1 / S8)

@pytest.mark.parametrize("n", [1, 2, 3, 16, 81, 255, 625])
def test_pack_unpack_bit_exact(orc, hp, n):
    """vec_R / mat_R (Eq. D10) are byte/index work plus one multiply or divide
    by the same double sqrt(2) on both sides: bit-exact against the oracle."""
    import torch
    rng = np.random.default_rng(100 + n)
    X = herm(rng, n)
    sv = orc.pack(X)
    A = hp.unpack(torch.from_numpy(sv).cuda(), n).cpu().numpy().T       # column-major content
    assert np.array_equal(A, orc.unpack(sv, n))
    sv2 = hp.pack(torch.from_numpy(np.ascontiguousarray(X.T)).cuda()).cpu().numpy()
    assert np.array_equal(sv2, sv)


# ------------------------------------------------------------------ BASELINE.json configs

def test_config1_n16(orc, hp):
    w = workloads.make(1)
    sv = pack_all(orc, [b.X for b in w.blocks])
    got, _ = check_vs_oracle(orc, hp, w.sizes, sv)
    b = w.blocks[0]
    closed = orc.pack((b.Q * np.maximum(b.lam, 0)[None, :]) @ b.Q.conj().T)
    assert rel_err(got, closed) <= TOL * 16
    check_invariants(orc, hp, w.sizes, sv, got)


def test_config2_256x81(orc, hp):
    w = workloads.make(2)
    sv = pack_all(orc, [b.X for b in w.blocks])
    got, _ = check_vs_oracle(orc, hp, w.sizes, sv, nthreads=1)
    check_invariants(orc, hp, w.sizes, sv, got)


def test_config3_n625(orc, hp):
    w = workloads.make(3)
    sv = pack_all(orc, [b.X for b in w.blocks])
    got, _ = check_vs_oracle(orc, hp, w.sizes, sv, nthreads=orc.max_threads())
    b = w.blocks[0]
    closed = orc.pack((b.Q * np.maximum(b.lam, 0)[None, :]) @ b.Q.conj().T)
    assert rel_err(got, closed) <= TOL * 625
    check_invariants(orc, hp, w.sizes, sv, got)


def test_config4_mixed_full_size(orc, hp):
    """Full config 4 in ONE call (1296 + 2401 + 64 x 36): every block element by element against the oracle
    (the n = 2401 block, the only GUE-type matrix above n = 1296, takes the threaded oracle about a minute),
    then the library-independent KKT certificate."""
    w = workloads.make(4)
    sizes = w.sizes
    sv = pack_all(orc, [b.X for b in w.blocks])
    got = gpu_project(hp, sizes, sv)
    offs = np.concatenate([[0], np.cumsum([n * n for n in sizes])])
    worst = {}
    for k, n in enumerate(sizes):
        seg = sv[offs[k]:offs[k + 1]]
        want = orc.project([n], seg, nthreads=orc.max_threads() if n > 100 else 1)
        err = rel_err(got[offs[k]:offs[k + 1]], want)
        worst[n] = max(worst.get(n, 0.0), err)
        assert err <= TOL * n, (k, n, err)
    _record("config4 vs oracle", {str(k): v for k, v in worst.items()})
    err, nrm = check_oracle_samples(4, got)          # the stored oracle run of the whole config agrees as well
    assert err <= TOL * 2401 and nrm <= TOL * 2401, (err, nrm)
    check_invariants(orc, hp, sizes, sv, got)


def test_config4_permuted_block_order(orc, hp):
    """Block order must not matter: small blocks first, odd svec offsets."""
    rng = np.random.default_rng(44)
    sizes = [36, 81, 1, 129, 36, 0, 7, 200]
    mats = [herm(rng, n, 1 / np.sqrt(max(n, 1))) for n in sizes]
    sv = pack_all(orc, mats)
    got, _ = check_vs_oracle(orc, hp, sizes, sv)
    perm = [7, 3, 0, 5, 2, 6, 1, 4]
    sv_p = pack_all(orc, [mats[i] for i in perm])
    got_p = gpu_project(hp, [sizes[i] for i in perm], sv_p)
    offs = np.concatenate([[0], np.cumsum([n * n for n in sizes])])
    pos = 0
    for i in perm:
        n = sizes[i]
        assert np.array_equal(got_p[pos:pos + n * n], got[offs[i]:offs[i + 1]])   # same kernels, same bits
        pos += n * n


def test_config5_n4096_closed_form_and_invariants(orc, hp):
    """n = 4096 with 32-fold exactly repeated eigenvalues: the projection is still unique.  The
    oracle needs ~10 min on 8 cores, so the default run pins against the closed form from the
    generator's own Q and lambda (no eigensolver involved) and the invariants; HPSD_FULL_ORACLE=1
    adds the element-by-element oracle comparison."""
    w = workloads.make(5)
    b = w.blocks[0]
    sv = orc.pack(b.X)
    got = gpu_project(hp, [4096], sv)
    closed = orc.pack((b.Q * np.maximum(b.lam, 0)[None, :]) @ b.Q.conj().T)
    assert rel_err(got, closed) <= TOL * 4096
    check_invariants(orc, hp, [4096], sv, got)
    _record("config5 vs closed form", {"4096": rel_err(got, closed)})
    # the oracle itself at full size (14 minutes on 8 host cores): its stored samples, 8188 svec entries
    err, nrm = check_oracle_samples(5, got)
    _record("config5 vs oracle samples", {"4096": err})
    assert err <= TOL * 4096 and nrm <= TOL * 4096, (err, nrm)
    if os.environ.get("HPSD_FULL_ORACLE") == "1":
        want = orc.project([4096], sv, nthreads=orc.max_threads())
        err = rel_err(got, want)
        _record("config5 vs oracle", {"4096": err})
        assert err <= TOL * 4096


@pytest.mark.parametrize("n", [1891, 1930])
def test_panel_kernel_first_streamed_sizes_closed_form(orc, hp, n):
    """Sizes just above the resident limit of the panel kernel (12 tile slots x 148 SMs = 1776 tiles: n <= 1888):
    the first panels stream through the three-slot rings of the warp pairs with only one refill per ring, the last
    tile row is ragged (n is not a multiple of 32), later panels are resident.  Pinned against the closed form from
    the generator's own Q and lambda (no eigensolver) and the projection invariants."""
    rng = np.random.default_rng(workloads.BASE_SEED + 100 + n)
    b = workloads.from_spectrum(rng, workloads.spectrum_admm_lowrank(rng, n, n_big=8, sd=1e-1))
    sv = orc.pack(b.X)
    got = gpu_project(hp, [n], sv)
    closed = orc.pack((b.Q * np.maximum(b.lam, 0)[None, :]) @ b.Q.conj().T)
    assert rel_err(got, closed) <= TOL * n
    check_invariants(orc, hp, [n], sv, got)


# ------------------------------------------------------------------ sizes across both paths

@pytest.mark.parametrize("n", [2, 3, 4, 15, 31, 32, 33, 63, 64, 65, 83, 84])
def test_small_path_sizes(orc, hp, n):
    """S9: the Jacobi kernel on every size it supports (2..84)."""
    rng = np.random.default_rng(200 + n)
    sizes = [n] * 3
    sv = pack_all(orc, [herm(rng, n) for _ in sizes])
    hp.set_option("jacobi_max_n", 84)
    try:
        got, _ = check_vs_oracle(orc, hp, sizes, sv)
        check_invariants(orc, hp, sizes, sv, got)
    finally:
        hp.set_option("jacobi_max_n", 32)


@pytest.mark.parametrize("n", [33, 36, 47, 64, 65, 81, 83, 84, 100, 115, 116])
def test_medium_path_sizes(orc, hp, n):
    """S10 (default route for 32 < n <= 116): batched divide & conquer up to n = 83, in-CTA QL above."""
    rng = np.random.default_rng(250 + n)
    sizes = [n] * 3
    sv = pack_all(orc, [herm(rng, n) for _ in sizes])
    hp.set_option("medium_reroute", 0)          # keep the one-CTA kernels on the path (3 blocks of 84..116 would be rerouted)
    try:
        got, _ = check_vs_oracle(orc, hp, sizes, sv)
        check_invariants(orc, hp, sizes, sv, got)
    finally:
        hp.set_option("medium_reroute", 1)
    rerouted, _ = check_vs_oracle(orc, hp, sizes, sv)  # default dispatch (large path for few blocks of 84..116)
    assert rel_err(rerouted, got) <= TOL * n


@pytest.mark.parametrize("n,count", [(33, 1), (36, 5), (64, 2), (81, 7), (83, 1)])
def test_medium_path_in_cta_ql(orc, hp, n, count):
    """The in-CTA QL variant of S10 on sizes the batched D&C normally takes (option medium_dc = 0), and batch
    counts that are not powers of two for the D&C variant (the batch is padded with zero matrices)."""
    rng = np.random.default_rng(260 + n)
    sizes = [n] * count
    sv = pack_all(orc, [herm(rng, n) for _ in sizes])
    hp.set_option("medium_reroute", 0)
    try:
        got_dc, _ = check_vs_oracle(orc, hp, sizes, sv)
        hp.set_option("medium_dc", 0)
        got_ql, _ = check_vs_oracle(orc, hp, sizes, sv)
    finally:
        hp.set_option("medium_dc", 1)
        hp.set_option("medium_reroute", 1)
    assert rel_err(got_ql, got_dc) <= TOL * n


@pytest.mark.parametrize("n", [2, 5, 16, 31])
def test_medium_kernel_on_small_sizes(orc, hp, n):
    """The S10 kernels have no lower size limit: route small blocks through them (D&C with a single leaf)."""
    rng = np.random.default_rng(270 + n)
    sizes = [n] * 2
    sv = pack_all(orc, [herm(rng, n) for _ in sizes])
    hp.set_option("jacobi_max_n", 1)
    try:
        check_vs_oracle(orc, hp, sizes, sv)
    finally:
        hp.set_option("jacobi_max_n", 32)


@pytest.mark.parametrize("cluster", [1, 0])
@pytest.mark.parametrize("n", [2, 3, 31, 32, 33, 63, 64, 65, 85, 96, 127, 128, 129, 200, 257, 320])
def test_large_path_sizes(orc, hp, n, cluster):
    """Force every block through S1..S8 of the Householder/D&C path (ragged tiles, several panels): with the
    cluster-resident reduction (default for 16 <= n <= 631) and with the grid-wide panel kernel (cluster = 0), which
    otherwise only serves n > 631."""
    rng = np.random.default_rng(300 + n)
    sv = orc.pack(herm(rng, n))
    force_large(hp, True)
    hp.set_option("cluster_tridiag", cluster)
    try:
        got, _ = check_vs_oracle(orc, hp, [n], sv, nthreads=orc.max_threads() if n > 150 else 1)
        check_invariants(orc, hp, [n], sv, got)
    finally:
        force_large(hp, False)
        hp.set_option("cluster_tridiag", 1)


# ------------------------------------------------------------------ two-stage reduction (S2 dense -> band, S3 bulge chasing, Q2)

TS_SIZES = [96, 97, 127, 128, 129, 160, 200, 257, 320, 449, 625]


def _band_to_dense(band, n, b):
    B = np.zeros((n, n), complex)
    for t in range(min(2 * b, n)):
        idx = np.arange(n - t)
        B[idx + t, idx] = band[:n - t, t]
    return B + np.tril(B, -1).conj().T


@pytest.mark.parametrize("n", TS_SIZES + [1296])
def test_two_stage_band_reduction(orc, hp, n):
    """S2 alone (hpsd_reduce_to_band): the band matrix is unitarily similar to the input (eigenvalues against numpy's
    eigvalsh of the input, a third opinion), Hermitian with a real diagonal, and nothing is stored
    outside the band width (rows b+1.. of the band storage are the bulge area of S3 and must be zero)."""
    import torch
    rng = np.random.default_rng(700 + n)
    X = herm(rng, n, 1 / np.sqrt(n))
    b = hp.band_width()
    band = hp.reduce_to_band(torch.from_numpy(orc.pack(X)).cuda(), n).cpu().numpy()
    assert np.abs(band[:, b + 1:]).max() == 0.0
    assert np.abs(band[:, 0].imag).max() == 0.0
    lam = np.linalg.eigvalsh(X)
    lb = np.linalg.eigvalsh(_band_to_dense(band, n, b))
    assert np.abs(lb - lam).max() <= 50 * n * EPS * np.abs(lam).max()
    assert abs(np.linalg.norm(band[:, 0]) ** 2 + 2 * np.linalg.norm(band[:, 1:]) ** 2 - np.linalg.norm(X) ** 2) <= 1e-12 * n * np.linalg.norm(X) ** 2


@pytest.mark.parametrize("n", TS_SIZES + [1296])
def test_two_stage_tridiagonal(orc, hp, n):
    """S2 + S3 (option two_stage = 1): the REAL tridiagonal (d, e) has the eigenvalues of the input."""
    import torch
    rng = np.random.default_rng(720 + n)
    X = herm(rng, n, 1 / np.sqrt(n))
    hp.set_option("two_stage", 1)
    try:
        d, e = hp.tridiagonalize(torch.from_numpy(orc.pack(X)).cuda(), n)
        d, e = d.cpu().numpy(), e.cpu().numpy()
    finally:
        hp.set_option("two_stage", 0)
    lam = np.linalg.eigvalsh(X)
    lt = np.linalg.eigvalsh(np.diag(d) + np.diag(e, 1) + np.diag(e, -1))
    assert np.abs(lt - lam).max() <= 50 * n * EPS * np.abs(lam).max()


@pytest.mark.parametrize("n", TS_SIZES)
def test_two_stage_whole_path(orc, hp, n):
    """The whole projection through S2 (band) + S3 (bulge chasing) + S4 + Q2 + Q1 + HERK against the oracle, and
    against the one-stage route of the same block."""
    rng = np.random.default_rng(740 + n)
    sv = orc.pack(herm(rng, n))
    force_large(hp, True)
    try:
        one = gpu_project(hp, [n], sv)
        hp.set_option("two_stage", 1)
        got, _ = check_vs_oracle(orc, hp, [n], sv, nthreads=orc.max_threads() if n > 150 else 1)
        check_invariants(orc, hp, [n], sv, got)
        assert rel_err(got, one) <= TOL * n
    finally:
        hp.set_option("two_stage", 0)
        force_large(hp, False)


def test_two_stage_in_a_mixed_cone_list(orc, hp):
    """Option two_stage = 2 (by size): in one call the blocks of at least two_stage_min_n rows take S2 + S3 + Q2, the
    others keep their routes (Jacobi, medium, cluster kernel); every block against the oracle, and the fused ADMM step."""
    import torch
    rng = np.random.default_rng(777)
    sizes = [150, 36, 260, 1, 16, 200]
    mats = [herm(rng, n, 1 / np.sqrt(max(n, 1))) for n in sizes]
    sv = pack_all(orc, mats)
    hp.set_option("two_stage", 2)
    hp.set_option("two_stage_min_n", 200)
    try:
        got, _ = check_vs_oracle(orc, hp, sizes, sv, nthreads=orc.max_threads())
        check_invariants(orc, hp, sizes, sv, got)
        v = pack_all(orc, [herm(rng, n, 0.1) for n in sizes])
        want_u, want_v = orc.admm_step(sizes, sv, v, nthreads=orc.max_threads())
        t_ut, t_v = torch.from_numpy(sv).cuda(), torch.from_numpy(v.copy()).cuda()
        t_u = torch.empty_like(t_ut)
        hp.admm_step_(sizes, t_ut, t_v, t_u)
        torch.cuda.synchronize()
        assert rel_err(t_u.cpu().numpy(), want_u) <= TOL * max(sizes)
        assert rel_err(t_v.cpu().numpy(), want_v) <= TOL * max(sizes)
    finally:
        hp.set_option("two_stage", 0)
        hp.set_option("two_stage_min_n", 1024)


@pytest.mark.parametrize("n", [150, 300])
def test_two_stage_degenerate_inputs(orc, hp, n):
    """Edge cases of the method on the two-stage route: already banded / tridiagonal / diagonal input (every
    reflector is trivial), rank one, exactly repeated eigenvalues, zero."""
    rng = np.random.default_rng(760 + n)
    force_large(hp, True)
    hp.set_option("two_stage", 1)
    try:
        for name, X in _special_cases(rng, n).items():
            X = 0.5 * (X + X.conj().T)
            sv = orc.pack(X)
            got = gpu_project(hp, [n], sv)
            want = orc.project([n], sv, nthreads=orc.max_threads())
            assert parity_err(got, want, sv, n) <= TOL * n, name
    finally:
        hp.set_option("two_stage", 0)
        force_large(hp, False)


@pytest.mark.parametrize("n", [1296, 2401])
def test_two_stage_config_sizes_closed_form(orc, hp, n):
    """Paper sizes d = 6, 7 on the two-stage route against the closed form from the generator's own Q and lambda
    (no eigensolver involved) and the library-independent KKT certificate."""
    rng = np.random.default_rng(workloads.BASE_SEED + 300 + n)
    b = workloads.from_spectrum(rng, workloads.spectrum_admm_lowrank(rng, n, n_big=8, sd=1e-1))
    sv = orc.pack(b.X)
    hp.set_option("two_stage", 1)
    try:
        got = gpu_project(hp, [n], sv)
        closed = orc.pack((b.Q * np.maximum(b.lam, 0)[None, :]) @ b.Q.conj().T)
        err = rel_err(got, closed)
        _record("two-stage vs closed form", {str(n): err})
        assert err <= TOL * n
        check_invariants(orc, hp, [n], sv, got)
    finally:
        hp.set_option("two_stage", 0)


# ------------------------------------------------------------------ non-finite input

@pytest.mark.parametrize("n,route", [(16, "jacobi"), (40, "meddc"), (100, "hhql"), (150, "cluster"), (150, "panel"), (150, "two_stage")])
@pytest.mark.parametrize("bad", [np.nan, np.inf, -np.inf])
def test_nonfinite_input_gives_nan_block(orc, hp, n, route, bad):
    """include/hpsd.h: a block with a NaN/Inf entry gets an all-NaN output block and info = 2; its neighbours in
    the same call are projected as usual (the paper is silent on non-finite input, DESIGN.md readings)."""
    import torch
    rng = np.random.default_rng(900 + n)
    mats = [herm(rng, n), herm(rng, n), herm(rng, 5)]
    sv = pack_all(orc, mats)
    sizes = [n, n, 5]
    clean = sv.copy()
    sv[n * n + (n * n) // 3] = bad                        # somewhere inside block 1
    hp.set_option("medium_reroute", 0)
    if route in ("cluster", "panel", "two_stage"):
        force_large(hp, True)
        hp.set_option("jacobi_max_n", 8)                  # the 5 x 5 neighbour stays on the Jacobi kernel
    if route == "panel":
        hp.set_option("cluster_tridiag", 0)
    if route == "two_stage":
        hp.set_option("two_stage", 1)
    try:
        t = torch.from_numpy(sv).cuda()
        ws = torch.empty(hp.workspace_size(sizes), dtype=torch.uint8, device="cuda")
        info = torch.zeros(len(sizes), dtype=torch.int32, device="cuda")
        out = torch.empty_like(t)
        hp.project_ws(sizes, t, out, ws, info=info)
        torch.cuda.synchronize()
        got, inf = out.cpu().numpy(), info.cpu().numpy()
        want = orc.project(sizes, clean)
    finally:
        force_large(hp, False)
        hp.set_option("medium_reroute", 1)
        hp.set_option("cluster_tridiag", 1)
        hp.set_option("two_stage", 0)
    assert np.isnan(got[n * n:2 * n * n]).all()
    assert list(inf) == [0, 2, 0]
    assert rel_err(got[:n * n], want[:n * n]) <= TOL * n
    assert rel_err(got[2 * n * n:], want[2 * n * n:]) <= TOL * n


# ------------------------------------------------------------------ degenerate inputs

def _special_cases(rng, n):
    v = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    G = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    psd = G @ G.conj().T / n
    lowrank = (G[:, :3] @ G[:, :3].conj().T) - (G[:, 3:5] @ G[:, 3:5].conj().T)
    Q, _ = np.linalg.qr(G)
    rep = np.repeat([-1.0, 0.5, 0.5, 2.0], [n - 3 * (n // 4), n // 4, n // 4, n // 4])[:n]
    return {
        "zero": np.zeros((n, n), complex),
        "diagonal": np.diag(rng.standard_normal(n)).astype(complex),
        "identity": np.eye(n, dtype=complex) * 1.5,
        "minus_identity": -np.eye(n, dtype=complex) * 0.5,
        "psd": psd,
        "nsd": -psd,
        "rank_one_plus": np.outer(v, v.conj()),
        "rank_one_minus": -np.outer(v, v.conj()),
        "low_rank_indefinite": lowrank,
        "repeated_eigenvalues": (Q * rep[None, :]) @ Q.conj().T,
        "tiny_scale": herm(rng, n) * 1e-100,
        "huge_scale": herm(rng, n) * 1e100,
        "tridiagonal_already": np.diag(rng.standard_normal(n)).astype(complex)
        + np.diag(rng.standard_normal(n - 1), 1) + np.diag(rng.standard_normal(n - 1), 1).T,
        "block_diagonal": np.block([[herm(rng, n // 2), np.zeros((n // 2, n - n // 2))],
                                    [np.zeros((n - n // 2, n // 2)), herm(rng, n - n // 2)]]),
    }


@pytest.mark.parametrize("n,large", [(24, False), (24, True), (81, False), (150, True)])
def test_degenerate_inputs(orc, hp, n, large):
    rng = np.random.default_rng(500 + n)
    cases = _special_cases(rng, n)
    if large:
        force_large(hp, True)
    else:
        hp.set_option("medium_reroute", 0)      # keep the one-CTA kernels on the path (a single n = 81 block would be re-routed)
    try:
        for name, X in cases.items():
            X = 0.5 * (X + X.conj().T)
            sv = orc.pack(X)
            got = gpu_project(hp, [n], sv)
            want = orc.project([n], sv, nthreads=orc.max_threads() if n > 100 else 1)
            err = parity_err(got, want, sv, n)
            assert err <= TOL * n, (name, err)
            if name in ("zero", "minus_identity", "nsd", "rank_one_minus"):
                assert np.linalg.norm(got) <= TOL * n * max(np.linalg.norm(sv), 1e-300), name
            if name in ("diagonal", "identity"):       # closed form: clamp the diagonal
                np.testing.assert_allclose(got, np.maximum(sv, 0), rtol=8 * EPS, atol=0, err_msg=name)
    finally:
        force_large(hp, False)
        hp.set_option("medium_reroute", 1)


def test_n0_n1_and_empty_list(orc, hp):
    import torch
    out = hp.project([], torch.zeros(0, dtype=torch.float64, device="cuda"))
    assert out.numel() == 0
    sizes = [1, 0, 1, 1, 0]
    sv = np.array([2.5, -3.0, 0.0])
    got = gpu_project(hp, sizes, sv)
    assert np.array_equal(got, np.array([2.5, 0.0, 0.0]))
    assert np.array_equal(got, orc.project(sizes, sv))


def test_in_place_call(orc, hp):
    """in_svec == out_svec is allowed (include/hpsd.h): both paths, mixed list."""
    import torch
    rng = np.random.default_rng(7)
    sizes = [40, 150, 1, 12]
    sv = pack_all(orc, [herm(rng, n) for n in sizes])
    ref = gpu_project(hp, sizes, sv)
    t = torch.from_numpy(sv.copy()).cuda()
    hp.project_(sizes, t, t)
    torch.cuda.synchronize()
    assert np.array_equal(t.cpu().numpy(), ref)


def test_caller_workspace_info_and_errors(orc, hp):
    import torch
    rng = np.random.default_rng(8)
    sizes = [30, 140]
    sv = pack_all(orc, [herm(rng, n) for n in sizes])
    need = hp.workspace_size(sizes)
    assert need > 0
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    info = torch.full((2,), 77, dtype=torch.int32, device="cuda")
    t = torch.from_numpy(sv).cuda()
    out = torch.empty_like(t)
    hp.project_ws(sizes, t, out, ws, info)
    torch.cuda.synchronize()
    assert info.cpu().tolist() == [0, 0]
    assert np.array_equal(out.cpu().numpy(), gpu_project(hp, sizes, sv))
    with pytest.raises(hp.HpsdError, match="workspace"):
        hp.project_ws(sizes, t, out, ws[: need // 2], info)
    lib = hp.load_library()
    import ctypes
    arr = (ctypes.c_int * 1)(-3)
    assert lib.hpsd_project(1, arr, t.data_ptr(), out.data_ptr(), None) == -1          # HPSD_EINVAL
    assert lib.hpsd_project(-1, arr, t.data_ptr(), out.data_ptr(), None) == -1
    arr = (ctypes.c_int * 1)(5)
    assert lib.hpsd_project(1, arr, None, out.data_ptr(), None) == -1


def test_project_host_roundtrip(orc, hp):
    """hpsd_project_host (the e2e call bench.py times): host buffers in and out."""
    import torch
    rng = np.random.default_rng(9)
    sizes = [20, 100]
    sv = pack_all(orc, [herm(rng, n) for n in sizes])
    h_in = torch.from_numpy(sv).pin_memory()
    h_out = hp.project_host(sizes, h_in)
    assert np.array_equal(h_out.numpy(), gpu_project(hp, sizes, sv))


def test_stream_and_graph_capture(orc, hp):
    """The call only enqueues on the caller's stream and is capturable in a CUDA graph once the plan
    and workspace exist (include/hpsd.h conventions)."""
    import torch
    rng = np.random.default_rng(10)
    sizes = [16, 130]
    sv = pack_all(orc, [herm(rng, n) for n in sizes])
    ref = gpu_project(hp, sizes, sv)          # creates plan + workspace
    t = torch.from_numpy(sv).cuda()
    out = torch.zeros_like(t)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        hp.project_(sizes, t, out)            # warm-up on the side stream
    s.synchronize()
    g = torch.cuda.CUDAGraph()
    out.zero_()
    with torch.cuda.graph(g, stream=s):
        hp.project_(sizes, t, out)
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), ref)


def test_eigvalsh_and_tridiagonalize(orc, hp):
    """S2+S3 alone and S2..S4 alone: eigenvalues against the oracle's (sorted)."""
    import torch
    for n in (2, 50, 200):
        rng = np.random.default_rng(600 + n)
        X = herm(rng, n)
        sv = orc.pack(X)
        lam_o, _ = orc.eigh_svec(sv, n)
        lam_o = np.sort(lam_o)
        t = torch.from_numpy(sv).cuda()
        lam = hp.eigvalsh(t, n).cpu().numpy()
        assert np.all(np.diff(lam) >= 0)
        assert np.abs(lam - lam_o).max() <= TOL * n * np.abs(lam_o).max()
        d, e = hp.tridiagonalize(t, n)
        d, e = d.cpu().numpy(), e.cpu().numpy()
        T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
        # similarity invariants: trace and Frobenius norm
        assert abs(d.sum() - np.trace(X).real) <= TOL * n * np.linalg.norm(X)
        assert abs(np.linalg.norm(T) - np.linalg.norm(X)) <= TOL * n * np.linalg.norm(X)


def test_covariances(orc, hp):
    """P(alpha X) = alpha P(X) for alpha = 2^k (exact in floating point); conjugation covariance
    P(conj X) = conj P(X), which is why the triangle/sign convention of (D10) does not matter
    (SURVEY.md §8(b))."""
    rng = np.random.default_rng(11)
    for n, force in ((40, False), (140, True)):
        if force:
            force_large(hp, True)
        try:
            X = herm(rng, n)
            sv = orc.pack(X)
            p = gpu_project(hp, [n], sv)
            assert np.array_equal(gpu_project(hp, [n], 4.0 * sv), 4.0 * p)
            pc = gpu_project(hp, [n], orc.pack(X.conj()))
            assert rel_err(pc, orc.pack(orc.unpack(p, n).conj())) <= TOL * n
        finally:
            force_large(hp, False)


def test_admm_step_fused(orc, hp):
    """NEXT-2: u = Pi_C(u~ - v), v <- v - u~ + u (Eqs. D33-D34) fused into
    S1 and S8, against the oracle's unfused version; every size class in one list; u aliasing u~."""
    import torch
    rng = np.random.default_rng(12)
    sizes = [1, 24, 81, 150, 1, 36]
    ut = pack_all(orc, [herm(rng, n) for n in sizes])
    v = pack_all(orc, [herm(rng, n) for n in sizes])
    want_u, want_v = orc.admm_step(sizes, ut, v, nthreads=orc.max_threads())
    t_ut, t_v = torch.from_numpy(ut).cuda(), torch.from_numpy(v.copy()).cuda()
    t_u = torch.empty_like(t_ut)
    hp.admm_step_(sizes, t_ut, t_v, t_u)
    torch.cuda.synchronize()
    off = 0
    for n in sizes:
        sl = slice(off, off + n * n)
        assert parity_err(t_u.cpu().numpy()[sl], want_u[sl], (ut - v)[sl], n) <= TOL * n, n
        assert parity_err(t_v.cpu().numpy()[sl], want_v[sl], (ut - v)[sl], n) <= TOL * n, n
        off += n * n
    # the plain projection of the difference gives the same u bit for bit (same kernels, same arithmetic)
    assert np.array_equal(t_u.cpu().numpy(), gpu_project(hp, sizes, (torch.from_numpy(ut) - torch.from_numpy(v)).numpy()))
    # in place: u written over u~
    t_ut2, t_v2 = torch.from_numpy(ut.copy()).cuda(), torch.from_numpy(v.copy()).cuda()
    hp.admm_step_(sizes, t_ut2, t_v2, t_ut2)
    torch.cuda.synchronize()
    assert np.array_equal(t_ut2.cpu().numpy(), t_u.cpu().numpy())
    assert np.array_equal(t_v2.cpu().numpy(), t_v.cpu().numpy())


@pytest.mark.parametrize("n", [117, 130, 255, 256, 257, 400, 625, 631])
def test_cluster_tridiag_kernel(orc, hp, n):
    """S1+S2+S3 by the cluster-resident kernel (tridiag_cluster.cu; option "cluster_tridiag", on by default).
    Whole-path parity against the oracle, (d, e) against the grid-wide panel kernel (same reflector convention,
    so the tridiagonals agree to rounding), and the fused ADMM subtraction of Eq. (D33) on this path."""
    import torch
    rng = np.random.default_rng(700 + n)
    sv = orc.pack(herm(rng, n, 1.0 / np.sqrt(n)))
    t = torch.from_numpy(sv).cuda()
    hp.set_option("cluster_tridiag", 0)
    d0, e0 = hp.tridiagonalize(t, n)
    hp.set_option("cluster_tridiag", 1)
    try:
        got, _ = check_vs_oracle(orc, hp, [n], sv, nthreads=orc.max_threads())
        d1, e1 = hp.tridiagonalize(t, n)
        v = orc.pack(herm(rng, n, 1.0 / np.sqrt(n)))
        t_v, t_u = torch.from_numpy(v.copy()).cuda(), torch.empty_like(t)
        hp.admm_step_([n], t, t_v, t_u)
        torch.cuda.synchronize()
        want_u, want_v = orc.admm_step([n], sv, v, nthreads=orc.max_threads())
    finally:
        hp.set_option("cluster_tridiag", 1)
    scale = float(d0.abs().max() + e0.abs().max())
    assert float((d1 - d0).abs().max()) <= 1e-13 * n * scale
    assert float((e1 - e0).abs().max()) <= 1e-13 * n * scale
    assert parity_err(t_u.cpu().numpy(), want_u, sv - v, n) <= TOL * n
    assert parity_err(t_v.cpu().numpy(), want_v, sv - v, n) <= TOL * n


def test_graph_replay_of_repeated_calls(orc, hp):
    """Option "graph_replay" (default 1): the second and later calls with the same size list and the same buffers
    (an ADMM loop) are replayed as a CUDA graph.  The replay must equal the plain launches bit for bit, must see new
    CONTENTS of the same buffers, must work on a non-default stream, and the fused ADMM step must replay as well."""
    import torch
    rng = np.random.default_rng(77)
    sizes = [150, 1, 24, 81, 36]
    sv1 = pack_all(orc, [herm(rng, n) for n in sizes])
    sv2 = pack_all(orc, [herm(rng, n) for n in sizes])
    hp.set_option("graph_replay", 0)
    plain1, plain2 = gpu_project(hp, sizes, sv1), gpu_project(hp, sizes, sv2)
    hp.set_option("graph_replay", 1)
    t_in, t_out = torch.from_numpy(sv1.copy()).cuda(), torch.empty(sv1.size, dtype=torch.float64, device="cuda")
    for it in range(4):                                  # 1: plain launches, 2: capture + launch, 3-4: replay
        t_out.zero_()
        hp.project_(sizes, t_in, t_out)
        torch.cuda.synchronize()
        assert np.array_equal(t_out.cpu().numpy(), plain1), it
    t_in.copy_(torch.from_numpy(sv2))                    # same buffers, new contents
    hp.project_(sizes, t_in, t_out)
    torch.cuda.synchronize()
    assert np.array_equal(t_out.cpu().numpy(), plain2)
    want = orc.project(sizes, sv2, nthreads=orc.max_threads())
    off = 0
    for n in sizes:
        sl = slice(off, off + n * n)
        assert parity_err(t_out.cpu().numpy()[sl], want[sl], sv2[sl], n) <= TOL * n
        off += n * n
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        for _ in range(3):
            hp.project_(sizes, t_in, t_out, stream=s)
    s.synchronize()
    assert np.array_equal(t_out.cpu().numpy(), plain2)
    # fused ADMM step (Eqs. D33-D34), repeated with the same buffers: v changes every iteration
    ut, v = torch.from_numpy(sv1.copy()).cuda(), torch.from_numpy(sv2.copy()).cuda()
    u = torch.empty_like(ut)
    v_ref, u_ref = sv2.copy(), None
    for it in range(3):
        hp.admm_step_(sizes, ut, v, u)
        torch.cuda.synchronize()
        u_ref, v_ref = orc.admm_step(sizes, sv1, v_ref, nthreads=orc.max_threads())
        assert rel_err(u.cpu().numpy(), u_ref) <= TOL * max(sizes), it
        assert rel_err(v.cpu().numpy(), v_ref) <= TOL * max(sizes), it


def test_concurrent_lanes_of_cluster_sized_blocks(orc, hp):
    """Option "large_lanes" (default 1): several blocks whose reduction runs on one 16-CTA cluster are processed next to
    each other on internal lane streams.  Must equal the sequential result BIT FOR BIT on every repetition (eight
    clusters of n = 625 at once once exposed a shared-memory aliasing race in the cluster kernel), through plain
    launches and graph replay, and match the oracle; plus a mixed list with sequential (n > 631) and small blocks."""
    import torch
    rng = np.random.default_rng(88)
    for n, count, reps in ((625, 8, 30), (116, 7, 10), (300, 3, 6)):
        sizes = [n] * count
        sv = pack_all(orc, [herm(rng, n, 1.0 / np.sqrt(n)) for _ in sizes])
        force_large(hp, True)                     # the same route with and without lanes (the re-routing rule depends on them)
        try:
            hp.set_option("large_lanes", 0)
            base = gpu_project(hp, sizes, sv)
            hp.set_option("large_lanes", 1)
            t_in = torch.from_numpy(sv).cuda()
            t_out = torch.empty_like(t_in)
            for it in range(reps):
                t_out.zero_()
                hp.project_(sizes, t_in, t_out)
                if it % 3 == 0:
                    torch.cuda.synchronize()
                assert np.array_equal(t_out.cpu().numpy(), base), (n, it)
        finally:
            force_large(hp, False)
            hp.set_option("large_lanes", 1)
        if n != 625:
            want = orc.project(sizes, sv, nthreads=orc.max_threads())
            assert rel_err(base, want) <= TOL * n
    sizes = [200, 700, 36, 150, 1, 36, 420]
    sv = pack_all(orc, [herm(rng, n, 1.0 / np.sqrt(max(n, 1))) for n in sizes])
    check_vs_oracle(orc, hp, sizes, sv, nthreads=orc.max_threads())


def test_panel_lanes_of_blocks_above_the_cluster_limit(orc, hp):
    """Option "panel_lanes" (default 1): two or more blocks that take the grid-wide cooperative panel kernel are dealt to two
    lanes on disjoint sets of SMs (lane 1: 64 CTAs on a library stream, forked behind an event inside lane 0's reduction;
    lane 0: the caller's stream, capped from that panel on).  The CTA count changes summation orders, so the result is
    compared with the oracle (and with the sequential schedule to rounding), must be identical on every repetition
    (plain launches, capture, graph replays) and must work through a caller-owned workspace."""
    import torch
    rng = np.random.default_rng(99)
    for sizes in ([700, 640], [800, 36, 650, 1, 900, 625], [1000, 700, 700, 660]):
        sv = pack_all(orc, [herm(rng, n, 1.0 / np.sqrt(max(n, 1))) for n in sizes])
        hp.set_option("panel_lanes", 0)
        try:
            base = gpu_project(hp, sizes, sv)
        finally:
            hp.set_option("panel_lanes", 1)
        got, want = check_vs_oracle(orc, hp, sizes, sv, nthreads=orc.max_threads())
        assert rel_err(got, base) <= 1e-13
        t_in = torch.from_numpy(sv).cuda()
        t_out = torch.empty_like(t_in)
        for it in range(5):
            t_out.zero_()
            hp.project_(sizes, t_in, t_out)
            assert np.array_equal(t_out.cpu().numpy(), got), (sizes, it)
        ws = torch.empty(hp.workspace_size(sizes), dtype=torch.uint8, device="cuda")
        info = torch.full((len(sizes),), -1, dtype=torch.int32, device="cuda")
        t_out.zero_()
        hp.project_ws(sizes, t_in, t_out, ws, info)
        torch.cuda.synchronize()
        assert info.cpu().tolist() == [0] * len(sizes)
        assert np.array_equal(t_out.cpu().numpy(), got)
    # caller-side capture: lane 1 joins the capture through the fork event inside lane 0's reduction and is joined at the end
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    t_in2, t_out2 = t_in.clone(), torch.zeros_like(t_in)
    with torch.cuda.stream(side):
        hp.project_(sizes, t_in2, t_out2)
    side.synchronize()
    g = torch.cuda.CUDAGraph()
    t_out2.zero_()
    with torch.cuda.graph(g, stream=side):
        hp.project_(sizes, t_in2, t_out2)
    for _ in range(2):
        t_out2.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(t_out2.cpu().numpy(), got)


def test_random_cone_lists(orc, hp):
    """Seeded random cone lists across every route (scalars, Jacobi, one-CTA medium kernels, re-routed medium blocks,
    cluster-sized blocks on lanes, panel-kernel blocks) and several matrix structures (dense, low-rank + noise, exact
    repeated eigenvalues, diagonal, scaled by 1e-8 .. 1e8): per-block parity with the oracle on the first call, on the
    captured call and on the graph replay."""
    import torch
    rng = np.random.default_rng(4242)

    def rand_size():
        k = rng.integers(0, 10)
        if k == 0:
            return 1
        if k <= 2:
            return int(rng.integers(2, 33))
        if k <= 4:
            return int(rng.integers(33, 117))
        if k <= 7:
            return int(rng.integers(117, 632))
        if k == 8:
            return int(rng.integers(632, 700))
        return int(rng.choice([16, 36, 81]))

    def rand_mat(n):
        kind = rng.integers(0, 5)
        h = herm(rng, n, 1.0 / np.sqrt(max(n, 1)))
        if kind == 0 or n < 3:
            return h
        if kind == 1:
            r = max(1, n // 20)
            b = rng.standard_normal((n, r)) + 1j * rng.standard_normal((n, r))
            return b @ b.conj().T / n + 1e-3 * h
        if kind == 2:
            q = workloads.haar_unitary(rng, n)
            lam = np.repeat(rng.standard_normal(n // 8 + 1), 8)[:n]
            x = (q * lam) @ q.conj().T
            return 0.5 * (x + x.conj().T)
        if kind == 3:
            return np.diag(rng.standard_normal(n)).astype(complex)
        return h * 10.0 ** int(rng.integers(-8, 9))

    for _ in range(12):
        sizes = [rand_size() for _ in range(int(rng.integers(1, 9)))]
        sv = pack_all(orc, [rand_mat(n) for n in sizes])
        want = orc.project(sizes, sv, nthreads=orc.max_threads())
        t_in = torch.from_numpy(sv).cuda()
        t_out = torch.empty_like(t_in)
        for rep in range(3):
            t_out.zero_()
            hp.project_(sizes, t_in, t_out)
            torch.cuda.synchronize()
            got, off = t_out.cpu().numpy(), 0
            for n in sizes:
                sl = slice(off, off + n * n)
                assert parity_err(got[sl], want[sl], sv[sl], n) <= TOL * max(n, 1), (sizes, n, rep)
                off += n * n


# ------------------------------------------------------------------ explicit plan handle, streams

def test_plan_api_admm_loop_under_capture(orc, hp):
    """hpsd_plan_create / execute / destroy.  One plan serves a 100-iteration ADMM cone-step loop
    (Eqs. D33-D34) captured by the CALLER into a CUDA graph; the iterates match the oracle's loop step by step for the
    first steps and the fixed point at the end (v_k converges: u = P(u~ - v), v <- v - u~ + u with constant u~
    gives v -> P(-(u~))-like limits; we simply compare against the oracle's own 100 steps)."""
    import torch
    rng = np.random.default_rng(31)
    sizes = [16, 36, 1, 150, 16]
    ut = pack_all(orc, [herm(rng, n) for n in sizes])
    v0 = pack_all(orc, [herm(rng, n) * 0.1 for n in sizes])
    plan = hp.Plan(sizes)
    try:
        assert plan.workspace_bytes() >= hp.workspace_size(sizes) - 4096
        t_ut, t_v, t_u = torch.from_numpy(ut).cuda(), torch.from_numpy(v0.copy()).cuda(), torch.empty(len(ut), dtype=torch.float64, device="cuda")
        # eager steps first (plain launches, then the library's own graph), checked against the oracle
        v = v0.copy()
        for _ in range(3):
            plan.admm_step_(t_ut, t_v, t_u)
            u, v = orc.admm_step(sizes, ut, v, nthreads=orc.max_threads())
        torch.cuda.synchronize()
        assert rel_err(t_u.cpu().numpy(), u) <= TOL * max(sizes)
        assert rel_err(t_v.cpu().numpy(), v) <= TOL * max(sizes)
        assert plan.info() == [0] * len(sizes)
        # caller-side capture of one step, replayed 97 times
        side = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            with torch.cuda.graph(g, stream=side):
                plan.admm_step_(t_ut, t_v, t_u, stream=side)
        for _ in range(97):
            g.replay()
            u, v = orc.admm_step(sizes, ut, v, nthreads=orc.max_threads())
        torch.cuda.synchronize()
        assert rel_err(t_u.cpu().numpy(), u) <= 100 * TOL * max(sizes)      # 100 steps of rounding in the v recursion
        assert rel_err(t_v.cpu().numpy(), v) <= 100 * TOL * max(sizes)
        # plain projection through the same plan
        out = torch.empty_like(t_ut)
        plan.project_(t_ut, out)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), gpu_project(hp, sizes, ut))
    finally:
        plan.destroy()


def test_plan_options_are_frozen_at_creation(orc, hp):
    """A plan keeps the options it was created with: changing a routing option afterwards does not alter its result
    bits, and a plan created under the new option takes the new route."""
    import torch
    rng = np.random.default_rng(32)
    n = 200
    sv = orc.pack(herm(rng, n))
    t = torch.from_numpy(sv).cuda()
    a = hp.Plan([n])
    out_a = a.project_(t, torch.empty_like(t)).cpu().numpy()
    hp.set_option("cluster_tridiag", 0)
    try:
        b = hp.Plan([n])
        out_a2 = a.project_(t, torch.empty_like(t)).cpu().numpy()
        out_b = b.project_(t, torch.empty_like(t)).cpu().numpy()
    finally:
        hp.set_option("cluster_tridiag", 1)
    assert np.array_equal(out_a, out_a2)
    assert not np.array_equal(out_a, out_b)                      # other kernels, other rounding
    want = orc.project([n], sv, nthreads=orc.max_threads())
    assert rel_err(out_a, want) <= TOL * n and rel_err(out_b, want) <= TOL * n
    a.destroy(); b.destroy()


def test_two_streams_share_the_library_workspace(orc, hp):
    """hpsd_project from two streams without host synchronisation in between: the calls share the library
    workspace and are ordered on it with an event, so both results are right; two explicit plans on two
    streams run independently."""
    import torch
    rng = np.random.default_rng(33)
    na, nb = 300, 310
    sva, svb = orc.pack(herm(rng, na)), orc.pack(herm(rng, nb))
    ta, tb = torch.from_numpy(sva).cuda(), torch.from_numpy(svb).cuda()
    oa, ob = torch.empty_like(ta), torch.empty_like(tb)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    for _ in range(5):
        hp.project_([na], ta, oa, stream=s1)
        hp.project_([nb], tb, ob, stream=s2)
    torch.cuda.synchronize()
    wa = orc.project([na], sva, nthreads=orc.max_threads())
    wb = orc.project([nb], svb, nthreads=orc.max_threads())
    assert rel_err(oa.cpu().numpy(), wa) <= TOL * na
    assert rel_err(ob.cpu().numpy(), wb) <= TOL * nb
    pa, pb = hp.Plan([na]), hp.Plan([nb])
    oa2, ob2 = torch.empty_like(ta), torch.empty_like(tb)
    for _ in range(5):
        pa.project_(ta, oa2, stream=s1)
        pb.project_(tb, ob2, stream=s2)
    torch.cuda.synchronize()
    assert np.array_equal(oa2.cpu().numpy(), oa.cpu().numpy())
    assert np.array_equal(ob2.cpu().numpy(), ob.cpu().numpy())
    pa.destroy(); pb.destroy()
