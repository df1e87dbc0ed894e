"""ctypes binding of the CPU oracle (oracle/hpsd_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs may import this.  It
imports nothing from paper_2606_20519_b200 and the product never imports it.

Every function cites the passage it follows in hpsd_oracle.c's header:
projection = eigendecomposition + zeroing negative eigenvalues
 on the vec_R encoding of Eq. (D10).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hpsd_oracle.c")
_LIB = os.path.join(_HERE, "libhpsd_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C99 + OpenMP).  Building the checker
    is not using it (__graft_entry__.build() calls this)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared",
               "-fno-fast-math", "-ffp-contract=off", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        vp = ctypes.c_void_p
        lib.orc_unpack.argtypes = [ctypes.c_int, dp, vp]
        lib.orc_unpack.restype = None
        lib.orc_pack.argtypes = [ctypes.c_int, vp, dp]
        lib.orc_pack.restype = None
        lib.orc_eigh_svec.argtypes = [ctypes.c_int, dp, dp, vp, ctypes.c_int]
        lib.orc_eigh_svec.restype = ctypes.c_int
        lib.orc_project_block.argtypes = [ctypes.c_int, dp, dp, ctypes.c_int]
        lib.orc_project_block.restype = ctypes.c_int
        lib.orc_project.argtypes = [ctypes.c_int, ip, dp, dp, ctypes.c_int]
        lib.orc_project.restype = ctypes.c_int
        lib.orc_max_threads.argtypes = []
        lib.orc_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def max_threads() -> int:
    return int(_load().orc_max_threads())


def svec_len(sizes: Sequence[int]) -> int:
    return int(sum(int(n) * int(n) for n in sizes))


def pack(X: np.ndarray) -> np.ndarray:
    """vec_R of Eq. (D10): Hermitian n x n -> n^2 doubles (lower triangle read)."""
    X = np.asarray(X, dtype=np.complex128)
    n = X.shape[0]
    assert X.shape == (n, n)
    a = np.asfortranarray(X)
    out = np.empty(n * n, dtype=np.float64)
    if n:
        _load().orc_pack(n, a.ctypes.data_as(ctypes.c_void_p), _dptr(out))
    return out


def unpack(sv: np.ndarray, n: int) -> np.ndarray:
    """mat_R, inverse of (D10): n^2 doubles -> full Hermitian n x n."""
    sv = np.ascontiguousarray(sv, dtype=np.float64)
    assert sv.shape == (n * n,)
    a = np.empty((n, n), dtype=np.complex128, order="F")
    if n:
        _load().orc_unpack(n, _dptr(sv), a.ctypes.data_as(ctypes.c_void_p))
    return a


def pack_blocks(mats: Sequence[np.ndarray]) -> np.ndarray:
    return np.concatenate([pack(m) for m in mats]) if len(mats) else np.zeros(0)


def unpack_blocks(sv: np.ndarray, sizes: Sequence[int]):
    out, off = [], 0
    for n in sizes:
        out.append(unpack(sv[off:off + n * n], n))
        off += n * n
    return out


def eigh_svec(sv: np.ndarray, n: int, nthreads: int = 1):
    """Eigenvalues (unsorted) and eigenvectors of one block given as svec."""
    sv = np.ascontiguousarray(sv, dtype=np.float64)
    lam = np.empty(n, dtype=np.float64)
    Z = np.empty((n, n), dtype=np.complex128, order="F")
    rc = _load().orc_eigh_svec(n, _dptr(sv), _dptr(lam), Z.ctypes.data_as(ctypes.c_void_p), nthreads)
    if rc != 0:
        raise RuntimeError(f"oracle QL did not converge (code {rc})")
    return lam, Z


def project(sizes: Sequence[int], in_svec: np.ndarray, nthreads: int = 1) -> np.ndarray:
    """Pi_C on a block list: svec in -> svec out."""
    sizes_a = np.ascontiguousarray(np.asarray(sizes, dtype=np.int32))
    x = np.ascontiguousarray(in_svec, dtype=np.float64)
    assert x.shape == (svec_len(sizes),), (x.shape, svec_len(sizes))
    out = np.empty_like(x)
    rc = _load().orc_project(len(sizes_a), sizes_a.ctypes.data_as(ctypes.POINTER(ctypes.c_int)),
                             _dptr(x), _dptr(out), nthreads)
    if rc != 0:
        raise RuntimeError(f"oracle projection failed (code {rc})")
    return out


def admm_step(sizes: Sequence[int], utilde: np.ndarray, v: np.ndarray, nthreads: int = 1):
    """The cone step of the SCS iteration exactly as the paper writes it, Eqs. (D33)-(D34)
    (PAPER.md:1466-1472):  u = Pi_C(u~ - v),  v_new = v - u~ + u.  Returns (u, v_new)."""
    utilde = np.ascontiguousarray(utilde, dtype=np.float64)
    v = np.ascontiguousarray(v, dtype=np.float64)
    u = project(sizes, utilde - v, nthreads=nthreads)
    return u, v - utilde + u
