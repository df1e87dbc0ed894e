"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/hpsd.h declares; argument errors are reported without a GPU; the product has no CPU
fallback and never touches oracle/."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_20519_b200 import build, binding
    build.build()
    return binding.load_library()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "hpsd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hpsd_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_all_exported(lib):
    from paper_2606_20519_b200 import binding
    names = declared_symbols()
    assert len(names) >= 14
    assert sorted(binding.EXPORTS) == names
    for name in names:
        assert getattr(lib, name) is not None, name


def test_version_and_strerror(lib):
    assert lib.hpsd_version() >= 100
    assert lib.hpsd_strerror(0) == b"success"
    assert b"argument" in lib.hpsd_strerror(-1)
    assert b"workspace" in lib.hpsd_strerror(-2)
    assert b"CUDA" in lib.hpsd_strerror(-3)
    assert lib.hpsd_strerror(-99) == b"unknown error"


def test_argument_errors_without_gpu(lib):
    bad = (ctypes.c_int * 2)(4, -1)
    sz = ctypes.c_size_t(0)
    assert lib.hpsd_workspace_size(2, bad, ctypes.byref(sz)) == -1
    assert lib.hpsd_workspace_size(-1, bad, ctypes.byref(sz)) == -1
    ok = (ctypes.c_int * 3)(16, 625, 36)
    assert lib.hpsd_workspace_size(3, ok, ctypes.byref(sz)) == 0
    assert sz.value > 16 * 625 * 625          # at least one complex copy of the large block
    small = (ctypes.c_int * 2)(16, 30)
    sz2 = ctypes.c_size_t(0)
    assert lib.hpsd_workspace_size(2, small, ctypes.byref(sz2)) == 0
    assert sz2.value < 4096                   # Jacobi blocks need no scratch, only the info words
    med = (ctypes.c_int * 3)(81, 81, 16)
    sz3 = ctypes.c_size_t(0)
    assert lib.hpsd_workspace_size(3, med, ctypes.byref(sz3)) == 0
    assert 16 * 2 * 81 * 81 < sz3.value < 5 << 20   # batched D&C scratch of the two n=81 blocks (or two large-path lanes)
    assert lib.hpsd_set_option(b"no_such_option", 1) == -1
    assert lib.hpsd_set_option(b"jacobi_max_n", 0) == -1
    assert lib.hpsd_set_option(b"jacobi_max_n", 84) == 0
    assert lib.hpsd_set_option(b"medium_max_n", 117) == -1
    assert lib.hpsd_set_option(b"medium_max_n", 116) == 0
    assert lib.hpsd_set_option(b"jacobi_max_n", 32) == 0
    assert lib.hpsd_project(0, None, None, None, None) == 0       # empty list: nothing to do


def test_no_cpu_fallback_without_device(lib):
    """Without a CUDA device every compute call fails loudly (include/hpsd.h)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    n = (ctypes.c_int * 1)(4)
    buf = (ctypes.c_double * 16)()
    assert lib.hpsd_project_host(1, n, buf, buf, None) < 0
    import paper_2606_20519_b200 as hp
    with pytest.raises(hp.HpsdError):
        hp.project([4], torch.zeros(16, dtype=torch.float64))


def test_product_never_imports_oracle():
    """oracle/ is test infrastructure: nothing under the package may import, link or run it."""
    pkg = os.path.join(ROOT, "paper_2606_20519_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "hpsd_oracle" not in txt and "libhpsd_oracle" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "hpsd_oracle.c")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_2606_20519_b200\b", otxt, flags=re.M)
    assert '#include "' not in otxt


def test_workspace_size_bounds_every_routing(lib):
    """hpsd_workspace_size is host-only and must bound every plan a device can make (include/hpsd.h, options
    "large_lanes", "panel_lanes", "medium_reroute"): lanes add one scratch area per concurrently processed cluster-sized
    block (up to 8), two or more blocks above the cluster limit run on two panel lanes (two areas), re-routed medium blocks
    need the large path's scratch, and switching the options off never needs more."""
    def ws(sizes):
        arr = (ctypes.c_int * len(sizes))(*sizes)
        sz = ctypes.c_size_t(0)
        assert lib.hpsd_workspace_size(len(sizes), arr, ctypes.byref(sz)) == 0
        return sz.value

    one = ws([625])
    assert ws([625, 625]) >= 2 * one - 4096                   # two lanes, two scratch areas
    assert ws([625] * 8) >= 8 * one - 8 * 4096
    assert ws([625] * 20) <= ws([625] * 8) + 4096             # at most 8 lanes
    assert ws([700, 700]) <= 2 * ws([700])                    # above the cluster limit: two panel lanes, two areas
    assert ws([700] * 5) <= ws([700, 700]) + 4096             # at most two panel lanes
    assert ws([4096, 4096]) < 1.5 * ws([4096])                # too large for panel lanes: one after the other, one area
    assert lib.hpsd_set_option(b"panel_lanes", 0) == 0
    try:
        assert ws([700, 700]) <= ws([700]) + 4096
    finally:
        assert lib.hpsd_set_option(b"panel_lanes", 1) == 0
    assert ws([100]) > 16 * 100 * 100                         # a single n = 100 block is re-routed to the large path
    assert lib.hpsd_set_option(b"large_lanes", 0) == 0
    assert lib.hpsd_set_option(b"panel_lanes", 0) == 0
    try:
        assert ws([625] * 8) <= ws([625]) + 4096
    finally:
        assert lib.hpsd_set_option(b"large_lanes", 1) == 0
        assert lib.hpsd_set_option(b"panel_lanes", 1) == 0
    assert lib.hpsd_set_option(b"medium_reroute", 0) == 0
    try:
        assert ws([100]) < 4096                               # the one-CTA kernel needs no scratch
    finally:
        assert lib.hpsd_set_option(b"medium_reroute", 1) == 0
