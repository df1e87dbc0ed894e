"""hpsd_project_static (include/hpsd.h): the allocation-free entry point, whose scratch is a fixed __device__ array of the
library.  Collected last on purpose (file name): the suite runs with pytest -x.

What is checked, through the C ABI:
  * two calls in a row (a full-size batch, then a smaller one that finds the first call's contents in the shared scratch,
    then the first again) against the EXISTING path hpsd_project on the same inputs, per block, at the tolerance of the
    parity tests (relative Frobenius error on the svec <= 1e-12 n), and one batch against the oracle;
  * sizes beyond the fixed capacity are rejected with HPSD_ETOOLARGE and nothing is written;
  * repeated calls leave the device's free memory where it was (no allocation on the call);
  * the non-finite contract (all-NaN block, info = 2) holds here too.
The test does not depend on what ran before it: it builds its own inputs and compares two paths of the same process."""
import numpy as np
import pytest

from conftest import rel_err

pytestmark = pytest.mark.gpu
TOL = 1e-12
HPSD_ETOOLARGE = -5


@pytest.fixture(scope="module")
def hp():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_20519_b200 as lib
    lib.load_library()
    return lib


def batch(orc, rng, n, count):
    """count random Hermitian n x n blocks (indefinite, O(1) spectrum) as one svec, blocks back to back."""
    out = []
    for _ in range(count):
        g = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
        out.append(orc.pack(0.5 * (g + g.conj().T) / np.sqrt(n)))
    return np.concatenate(out)


def compare(hp, n, count, sv_host):
    import torch
    sv = torch.from_numpy(sv_host).cuda()
    want = hp.project([n] * count, sv).cpu().numpy()          # existing path (plan, library workspace)
    got_t = torch.full_like(sv, float("nan"))
    info = torch.full((count,), -7, dtype=torch.int32, device="cuda")
    hp.project_static_(n, count, sv, got_t, info)
    torch.cuda.synchronize()
    got = got_t.cpu().numpy()
    assert info.cpu().tolist() == [0] * count
    for b in range(count):
        a, w = got[b * n * n:(b + 1) * n * n], want[b * n * n:(b + 1) * n * n]
        assert np.all(np.isfinite(a))
        assert rel_err(a, w) <= TOL * n, (n, count, b, rel_err(a, w))
    return got


def test_static_entry_matches_existing_path_on_calls_in_a_row(orc, hp):
    rng = np.random.default_rng(4242)
    big = batch(orc, rng, 81, 16)          # the paper's d = 3 block size, the largest batch the scratch takes
    small = batch(orc, rng, 36, 5)         # then a smaller batch on the same (now dirty) scratch
    first = compare(hp, 81, 16, big)
    compare(hp, 36, 5, small)
    again = compare(hp, 81, 16, big)
    assert np.array_equal(first, again)    # the stale contents of the scratch do not leak into the result
    compare(hp, 83, 16, batch(orc, rng, 83, 16))      # both limits at once
    compare(hp, 2, 1, batch(orc, rng, 2, 1))
    compare(hp, 16, 16, batch(orc, rng, 16, 16))      # hpsd_project takes the Jacobi kernel here: two algorithms agree
    # and against the oracle itself
    want = orc.project([81] * 3, big[:3 * 81 * 81])
    for b in range(3):
        s = slice(b * 6561, (b + 1) * 6561)
        assert rel_err(first[s], want[s]) <= TOL * 81


def test_static_entry_in_place_and_without_info(orc, hp):
    import torch
    rng = np.random.default_rng(4243)
    sv_host = batch(orc, rng, 64, 7)
    sv = torch.from_numpy(sv_host).cuda()
    want = hp.project([64] * 7, sv).cpu().numpy()
    hp.project_static_(64, 7, sv, sv)
    torch.cuda.synchronize()
    got = sv.cpu().numpy()
    for b in range(7):
        s = slice(b * 4096, (b + 1) * 4096)
        assert rel_err(got[s], want[s]) <= TOL * 64


def test_static_entry_rejects_sizes_beyond_its_capacity(hp):
    import torch
    lib = hp.load_library()
    buf = torch.zeros(17 * 84 * 84, dtype=torch.float64, device="cuda")
    out = torch.full_like(buf, 3.0)
    st = torch.cuda.current_stream().cuda_stream
    assert lib.hpsd_project_static(84, 1, buf.data_ptr(), out.data_ptr(), None, st) == HPSD_ETOOLARGE
    assert lib.hpsd_project_static(16, 17, buf.data_ptr(), out.data_ptr(), None, st) == HPSD_ETOOLARGE
    assert lib.hpsd_project_static(4096, 1, buf.data_ptr(), out.data_ptr(), None, st) == HPSD_ETOOLARGE
    assert lib.hpsd_project_static(1, 1, buf.data_ptr(), out.data_ptr(), None, st) == -1
    assert lib.hpsd_project_static(16, -1, buf.data_ptr(), out.data_ptr(), None, st) == -1
    assert lib.hpsd_project_static(16, 2, None, out.data_ptr(), None, st) == -1
    assert lib.hpsd_project_static(16, 0, None, None, None, st) == 0
    assert b"static scratch" in lib.hpsd_strerror(HPSD_ETOOLARGE)
    with pytest.raises(hp.HpsdError):
        hp.project_static_(84, 1, buf[:84 * 84], out[:84 * 84])
    torch.cuda.synchronize()
    assert bool((out == 3.0).all())        # a rejected call enqueues nothing


def test_static_entry_allocates_nothing(orc, hp):
    import torch
    rng = np.random.default_rng(4244)
    sv = torch.from_numpy(batch(orc, rng, 81, 16)).cuda()
    out = torch.empty_like(sv)
    hp.project_static_(81, 16, sv, out)     # first use on this device: kernel attributes, symbol address, module load
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(20):
        hp.project_static_(81, 16, sv, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0


def test_static_entry_non_finite_block(orc, hp):
    import torch
    rng = np.random.default_rng(4245)
    n, count = 40, 4
    sv_host = batch(orc, rng, n, count)
    sv_host[2 * n * n + 17] = np.inf
    sv = torch.from_numpy(sv_host).cuda()
    out = torch.empty_like(sv)
    info = torch.zeros(count, dtype=torch.int32, device="cuda")
    hp.project_static_(n, count, sv, out, info)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert info.cpu().tolist() == [0, 0, 2, 0]
    assert np.all(np.isnan(got[2 * n * n:3 * n * n]))
    want = hp.project([n] * count, sv).cpu().numpy()
    for b in (0, 1, 3):
        s = slice(b * n * n, (b + 1) * n * n)
        assert rel_err(got[s], want[s]) <= TOL * n
