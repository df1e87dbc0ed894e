"""ctypes binding of libhpsd.so -- argument marshalling only (names follow include/hpsd.h)."""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libhpsd.so")
_lib = None

# every symbol include/hpsd.h declares
EXPORTS = [
    "hpsd_version", "hpsd_strerror", "hpsd_project", "hpsd_workspace_size", "hpsd_project_ws",
    "hpsd_project_host", "hpsd_pack", "hpsd_unpack", "hpsd_tridiagonalize", "hpsd_eigvalsh",
    "hpsd_set_option", "hpsd_last_launch_count", "hpsd_release", "hpsd_fp64_peak_probe",
    "hpsd_profile_stage_count", "hpsd_profile_stage_name", "hpsd_profile_read", "hpsd_admm_step",
    "hpsd_reduce_to_band", "hpsd_band_width",
    "hpsd_plan_create", "hpsd_plan_destroy", "hpsd_plan_project", "hpsd_plan_admm_step", "hpsd_plan_info", "hpsd_plan_read_info", "hpsd_plan_host_overhead",
    "hpsd_project_approx", "hpsd_project_static",
    "hpsd_project_c64", "hpsd_admm_step_c64", "hpsd_plan_project_c64", "hpsd_plan_admm_step_c64", "hpsd_svec_convert",
    "hpsd_affine_create", "hpsd_affine_destroy", "hpsd_affine_dims", "hpsd_affine_apply_a", "hpsd_affine_apply_at", "hpsd_affine_project",
]


class HpsdError(RuntimeError):
    pass


def lib_path() -> str:
    return _LIB_PATH


def load_library():
    """Load libhpsd.so.  Fails loudly when the extension has not been built
    (python -m paper_2606_20519_b200.build, or __graft_entry__.build())."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise HpsdError(f"CUDA extension missing: {_LIB_PATH} (run __graft_entry__.build()); there is no CPU fallback")
        lib = ctypes.CDLL(_LIB_PATH)
        c_int, c_vp, c_sz = ctypes.c_int, ctypes.c_void_p, ctypes.c_size_t
        ip = ctypes.POINTER(ctypes.c_int)
        lib.hpsd_version.restype = c_int
        lib.hpsd_strerror.restype = ctypes.c_char_p
        lib.hpsd_strerror.argtypes = [c_int]
        lib.hpsd_project.argtypes = [c_int, ip, c_vp, c_vp, c_vp]
        lib.hpsd_admm_step.argtypes = [c_int, ip, c_vp, c_vp, c_vp, c_vp]
        lib.hpsd_workspace_size.argtypes = [c_int, ip, ctypes.POINTER(c_sz)]
        lib.hpsd_project_ws.argtypes = [c_int, ip, c_vp, c_vp, c_vp, c_sz, c_vp, c_vp]
        lib.hpsd_project_host.argtypes = [c_int, ip, c_vp, c_vp, c_vp]
        lib.hpsd_pack.argtypes = [c_int, c_vp, c_int, c_vp, c_vp]
        lib.hpsd_unpack.argtypes = [c_int, c_vp, c_vp, c_int, c_vp]
        lib.hpsd_tridiagonalize.argtypes = [c_int, c_vp, c_vp, c_vp, c_vp]
        lib.hpsd_eigvalsh.argtypes = [c_int, c_vp, c_vp, c_vp]
        lib.hpsd_reduce_to_band.argtypes = [c_int, c_vp, c_vp, c_vp]
        lib.hpsd_plan_create.argtypes = [c_int, ip, ctypes.POINTER(c_vp)]
        lib.hpsd_plan_destroy.argtypes = [c_vp]
        lib.hpsd_plan_project.argtypes = [c_vp, c_vp, c_vp, c_vp]
        lib.hpsd_plan_admm_step.argtypes = [c_vp, c_vp, c_vp, c_vp, c_vp]
        lib.hpsd_plan_info.argtypes = [c_vp, ctypes.POINTER(c_vp), ctypes.POINTER(c_sz)]
        lib.hpsd_plan_read_info.argtypes = [c_vp, ip, c_vp]
        lib.hpsd_plan_host_overhead.argtypes = [c_vp, c_vp, c_vp, c_int, c_vp, ctypes.POINTER(ctypes.c_double)]
        lib.hpsd_project_approx.argtypes = [c_int, c_vp, c_vp, c_int, c_vp]
        lib.hpsd_project_c64.argtypes = [c_int, ip, c_vp, c_vp, c_vp]
        lib.hpsd_admm_step_c64.argtypes = [c_int, ip, c_vp, c_vp, c_vp, c_vp]
        lib.hpsd_plan_project_c64.argtypes = [c_vp, c_vp, c_vp, c_vp]
        lib.hpsd_plan_admm_step_c64.argtypes = [c_vp, c_vp, c_vp, c_vp, c_vp]
        lib.hpsd_svec_convert.argtypes = [c_sz, c_vp, c_vp, c_int, c_vp]
        lib.hpsd_project_static.argtypes = [c_int, c_int, c_vp, c_vp, c_vp, c_vp]
        lib.hpsd_affine_create.argtypes = [c_int, ctypes.POINTER(c_vp)]
        lib.hpsd_affine_destroy.argtypes = [c_vp]
        lib.hpsd_affine_dims.argtypes = [c_vp, ip, ip]
        lib.hpsd_affine_apply_a.argtypes = [c_vp, c_vp, c_vp, c_vp]
        lib.hpsd_affine_apply_at.argtypes = [c_vp, c_vp, c_vp, c_vp]
        lib.hpsd_affine_project.argtypes = [c_vp, c_vp, c_vp, c_vp, c_vp, c_vp]
        lib.hpsd_set_option.argtypes = [ctypes.c_char_p, c_int]
        lib.hpsd_last_launch_count.restype = c_int
        lib.hpsd_release.restype = c_int
        lib.hpsd_fp64_peak_probe.argtypes = [c_int, c_int, ctypes.POINTER(ctypes.c_double), c_vp]
        lib.hpsd_profile_stage_name.restype = ctypes.c_char_p
        lib.hpsd_profile_stage_name.argtypes = [c_int]
        lib.hpsd_profile_read.argtypes = [ctypes.POINTER(ctypes.c_double), ip, c_int]
        for name in EXPORTS:
            if name not in ("hpsd_strerror", "hpsd_profile_stage_name"):
                getattr(lib, name).restype = getattr(lib, name).restype or c_int
        _lib = lib
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        msg = load_library().hpsd_strerror(rc).decode()
        raise HpsdError(f"{what} failed: {msg} (code {rc})")


def _sizes(sizes: Sequence[int]):
    arr = (ctypes.c_int * max(len(sizes), 1))(*[int(s) for s in sizes])
    return arr, len(sizes)


def _stream(stream: Optional[torch.cuda.Stream]) -> int:
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def _svec_suffix(*named) -> str:
    """"" for float64 svecs, "_c64" for float32 ones (complex64 storage, NEXT-1); all tensors of a call share the dtype."""
    dt = named[0][0].dtype
    if dt not in (torch.float64, torch.float32):
        raise HpsdError(f"{named[0][1]} must be a CUDA float64 (or float32: complex64 storage) tensor")
    for t, name in named:
        if not (t.is_cuda and t.dtype == dt and t.is_contiguous()):
            raise HpsdError(f"{name} must be a contiguous CUDA {dt} tensor")
    return "" if dt == torch.float64 else "_c64"


def _need_cuda_f64(t: torch.Tensor, name: str):
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise HpsdError(f"{name} must be a contiguous CUDA float64 tensor")


def svec_len(sizes: Sequence[int]) -> int:
    return int(sum(int(n) * int(n) for n in sizes))


def version() -> int:
    return int(load_library().hpsd_version())


def set_option(name: str, value: int) -> None:
    _check(load_library().hpsd_set_option(name.encode(), int(value)), "hpsd_set_option")


def last_launch_count() -> int:
    return int(load_library().hpsd_last_launch_count())


def release() -> None:
    _check(load_library().hpsd_release(), "hpsd_release")


def project_(sizes: Sequence[int], in_svec: torch.Tensor, out_svec: torch.Tensor,
             stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """hpsd_project: enqueue the projection of a cone list on `stream`; out may alias in."""
    lib = load_library()
    sfx = _svec_suffix((in_svec, "in_svec"), (out_svec, "out_svec"))
    total = svec_len(sizes)
    if in_svec.numel() != total or out_svec.numel() != total:
        raise HpsdError(f"svec length {in_svec.numel()}/{out_svec.numel()} != sum n^2 = {total}")
    arr, nb = _sizes(sizes)
    with torch.cuda.device(in_svec.device):
        _check(getattr(lib, "hpsd_project" + sfx)(nb, arr, in_svec.data_ptr(), out_svec.data_ptr(), _stream(stream)), "hpsd_project" + sfx)
    return out_svec


def project(sizes: Sequence[int], in_svec: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    return project_(sizes, in_svec, torch.empty_like(in_svec), stream)


def admm_step_(sizes: Sequence[int], utilde: torch.Tensor, v: torch.Tensor, u: torch.Tensor,
               stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """hpsd_admm_step: u = Pi_C(utilde - v), v <- v - utilde + u (v updated in place); returns u."""
    lib = load_library()
    sfx = _svec_suffix((utilde, "utilde"), (v, "v"), (u, "u"))
    total = svec_len(sizes)
    if utilde.numel() != total or v.numel() != total or u.numel() != total:
        raise HpsdError(f"svec lengths != sum n^2 = {total}")
    arr, nb = _sizes(sizes)
    with torch.cuda.device(utilde.device):
        _check(getattr(lib, "hpsd_admm_step" + sfx)(nb, arr, utilde.data_ptr(), v.data_ptr(), u.data_ptr(), _stream(stream)), "hpsd_admm_step" + sfx)
    return u


def workspace_size(sizes: Sequence[int]) -> int:
    arr, nb = _sizes(sizes)
    out = ctypes.c_size_t(0)
    _check(load_library().hpsd_workspace_size(nb, arr, ctypes.byref(out)), "hpsd_workspace_size")
    return int(out.value)


def project_ws(sizes: Sequence[int], in_svec: torch.Tensor, out_svec: torch.Tensor, ws: torch.Tensor,
               info: Optional[torch.Tensor] = None, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """hpsd_project_ws: caller-owned workspace (uint8 CUDA tensor) and optional int32 info[n_blocks]."""
    lib = load_library()
    _need_cuda_f64(in_svec, "in_svec")
    _need_cuda_f64(out_svec, "out_svec")
    if not (ws.is_cuda and ws.dtype == torch.uint8 and ws.is_contiguous()):
        raise HpsdError("ws must be a contiguous CUDA uint8 tensor")
    if info is not None and not (info.is_cuda and info.dtype == torch.int32 and info.numel() >= len(sizes)):
        raise HpsdError("info must be a CUDA int32 tensor with n_blocks entries")
    arr, nb = _sizes(sizes)
    with torch.cuda.device(in_svec.device):
        _check(lib.hpsd_project_ws(nb, arr, in_svec.data_ptr(), out_svec.data_ptr(), ws.data_ptr(), ws.numel(),
                                   info.data_ptr() if info is not None else None, _stream(stream)), "hpsd_project_ws")
    return out_svec


def project_host(sizes: Sequence[int], in_host: torch.Tensor, out_host: Optional[torch.Tensor] = None,
                 stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """hpsd_project_host: HOST float64 tensors in and out (pinned for async copies); synchronises."""
    lib = load_library()
    if in_host.is_cuda or in_host.dtype != torch.float64 or not in_host.is_contiguous():
        raise HpsdError("in_host must be a contiguous CPU float64 tensor")
    if out_host is None:
        out_host = torch.empty_like(in_host, pin_memory=in_host.is_pinned())
    arr, nb = _sizes(sizes)
    _check(lib.hpsd_project_host(nb, arr, in_host.data_ptr(), out_host.data_ptr(), _stream(stream)), "hpsd_project_host")
    return out_host


def pack(A: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """hpsd_pack: A is an (n, n) CUDA complex128 tensor holding the matrix in COLUMN-major order,
    i.e. A[j, i] in torch's row-major indexing is X_ij (pass X.T.contiguous())."""
    if not (A.is_cuda and A.dtype == torch.complex128 and A.is_contiguous() and A.dim() == 2 and A.shape[0] == A.shape[1]):
        raise HpsdError("A must be a contiguous square CUDA complex128 tensor (column-major content)")
    n = A.shape[0]
    out = torch.empty(n * n, dtype=torch.float64, device=A.device)
    with torch.cuda.device(A.device):
        _check(load_library().hpsd_pack(n, A.data_ptr(), n, out.data_ptr(), _stream(stream)), "hpsd_pack")
    return out


def unpack(svec: torch.Tensor, n: int, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """hpsd_unpack: returns an (n, n) complex128 tensor with column-major content (out[j, i] = X_ij)."""
    _need_cuda_f64(svec, "svec")
    if svec.numel() != n * n:
        raise HpsdError("svec length != n^2")
    out = torch.empty((n, n), dtype=torch.complex128, device=svec.device)
    with torch.cuda.device(svec.device):
        _check(load_library().hpsd_unpack(n, svec.data_ptr(), out.data_ptr(), n, _stream(stream)), "hpsd_unpack")
    return out


def tridiagonalize(svec: torch.Tensor, n: int, stream: Optional[torch.cuda.Stream] = None):
    _need_cuda_f64(svec, "svec")
    d = torch.empty(n, dtype=torch.float64, device=svec.device)
    e = torch.empty(max(n - 1, 0), dtype=torch.float64, device=svec.device)
    with torch.cuda.device(svec.device):
        _check(load_library().hpsd_tridiagonalize(n, svec.data_ptr(), d.data_ptr(), e.data_ptr(), _stream(stream)), "hpsd_tridiagonalize")
    return d, e


class Plan:
    """hpsd_plan_*: explicit plan handle (routing, options, workspace, status words and captured graphs of one size
    list).  Argument marshalling only; every step runs in the library's kernels."""

    def __init__(self, sizes: Sequence[int], device: Optional[torch.device] = None):
        self.sizes = [int(n) for n in sizes]
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self._h = ctypes.c_void_p()
        arr, nb = _sizes(self.sizes)
        with torch.cuda.device(self.device):
            _check(load_library().hpsd_plan_create(nb, arr, ctypes.byref(self._h)), "hpsd_plan_create")

    def project_(self, in_svec: torch.Tensor, out_svec: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
        sfx = _svec_suffix((in_svec, "in_svec"), (out_svec, "out_svec"))
        with torch.cuda.device(self.device):
            _check(getattr(load_library(), "hpsd_plan_project" + sfx)(self._h, in_svec.data_ptr(), out_svec.data_ptr(), _stream(stream)),
                   "hpsd_plan_project" + sfx)
        return out_svec

    def admm_step_(self, utilde: torch.Tensor, v: torch.Tensor, u: torch.Tensor, stream: Optional[torch.cuda.Stream] = None):
        sfx = _svec_suffix((utilde, "utilde"), (v, "v"), (u, "u"))
        with torch.cuda.device(self.device):
            _check(getattr(load_library(), "hpsd_plan_admm_step" + sfx)(self._h, utilde.data_ptr(), v.data_ptr(), u.data_ptr(), _stream(stream)),
                   "hpsd_plan_admm_step" + sfx)
        return u, v

    def info(self, stream: Optional[torch.cuda.Stream] = None):
        """hpsd_plan_read_info: status words of the last execution on `stream` as a list (synchronises the stream)."""
        nb = len(self.sizes)
        host = (ctypes.c_int * max(nb, 1))()
        with torch.cuda.device(self.device):
            _check(load_library().hpsd_plan_read_info(self._h, host, _stream(stream)), "hpsd_plan_read_info")
        return [int(host[i]) for i in range(nb)]

    def host_overhead_us(self, in_svec: torch.Tensor, out_svec: torch.Tensor, reps: int = 1000,
                         stream: Optional[torch.cuda.Stream] = None) -> float:
        """hpsd_plan_host_overhead: host microseconds per hpsd_plan_project call, measured inside the library."""
        us = ctypes.c_double()
        with torch.cuda.device(self.device):
            _check(load_library().hpsd_plan_host_overhead(self._h, in_svec.data_ptr(), out_svec.data_ptr(), int(reps), _stream(stream),
                                                          ctypes.byref(us)), "hpsd_plan_host_overhead")
        return float(us.value)

    def workspace_bytes(self) -> int:
        ptr, nbytes = ctypes.c_void_p(), ctypes.c_size_t()
        _check(load_library().hpsd_plan_info(self._h, ctypes.byref(ptr), ctypes.byref(nbytes)), "hpsd_plan_info")
        return int(nbytes.value)

    def destroy(self):
        if self._h:
            load_library().hpsd_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def project_approx(svec: torch.Tensor, n: int, iterations: int, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """hpsd_project_approx: composite-polynomial approximate projection of one block (NEXT-4)."""
    _need_cuda_f64(svec, "svec")
    if svec.numel() != n * n:
        raise HpsdError("svec length != n^2")
    out = torch.empty_like(svec)
    with torch.cuda.device(svec.device):
        _check(load_library().hpsd_project_approx(n, svec.data_ptr(), out.data_ptr(), int(iterations), _stream(stream)), "hpsd_project_approx")
    return out


def svec_convert(src: torch.Tensor, dtype: torch.dtype, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """hpsd_svec_convert: an svec between float64 and float32 storage (the single -> double switch of PAPER.md:1544)."""
    if not (src.is_cuda and src.is_contiguous() and {src.dtype, dtype} == {torch.float32, torch.float64}):
        raise HpsdError("svec_convert: contiguous CUDA tensor, float32 <-> float64")
    dst = torch.empty(src.shape, dtype=dtype, device=src.device)
    with torch.cuda.device(src.device):
        _check(load_library().hpsd_svec_convert(src.numel(), src.data_ptr(), dst.data_ptr(), 1 if dtype == torch.float32 else 0,
                                                _stream(stream)), "hpsd_svec_convert")
    return dst


def project_static_(n: int, count: int, in_svec: torch.Tensor, out_svec: torch.Tensor, info: Optional[torch.Tensor] = None,
                    stream: Optional[torch.cuda.Stream] = None) -> None:
    """hpsd_project_static: allocation-free exact projection of `count` blocks of one size n (n <= 83, count <= 16) on the
    library's fixed device scratch.  The caller passes input and output (and optionally an int32 status tensor); nothing is
    allocated here or in the library.  Calls that overlap on the GPU race on the scratch: keep them on one stream."""
    _need_cuda_f64(in_svec, "in_svec")
    _need_cuda_f64(out_svec, "out_svec")
    if in_svec.numel() != count * n * n or out_svec.numel() != count * n * n:
        raise HpsdError("svec length != count * n^2")
    ip = 0
    if info is not None:
        if not (info.is_cuda and info.dtype == torch.int32 and info.is_contiguous() and info.numel() >= count):
            raise HpsdError("info must be a contiguous CUDA int32 tensor of count entries")
        ip = info.data_ptr()
    with torch.cuda.device(in_svec.device):
        _check(load_library().hpsd_project_static(int(n), int(count), in_svec.data_ptr(), out_svec.data_ptr(), ip, _stream(stream)),
               "hpsd_project_static")


class Affine:
    """hpsd_affine_*: the affine-projection step of the SCS iteration (z_x = (a_x - A^T a_y)/2, z_y = a_y + A z_x) for
    the bipartite process-matrix SDP with local dimension d.  Argument marshalling only."""

    def __init__(self, d: int, device: Optional[torch.device] = None):
        self.d = int(d)
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self._h = ctypes.c_void_p()
        with torch.cuda.device(self.device):
            _check(load_library().hpsd_affine_create(self.d, ctypes.byref(self._h)), "hpsd_affine_create")
        n, m = ctypes.c_int(), ctypes.c_int()
        _check(load_library().hpsd_affine_dims(self._h, ctypes.byref(n), ctypes.byref(m)), "hpsd_affine_dims")
        self.n, self.m = int(n.value), int(m.value)

    def apply_A(self, x: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
        _need_cuda_f64(x, "x")
        y = torch.empty(self.n * self.n, dtype=torch.float64, device=x.device)
        with torch.cuda.device(self.device):
            _check(load_library().hpsd_affine_apply_a(self._h, x.data_ptr(), y.data_ptr(), _stream(stream)), "hpsd_affine_apply_a")
        return y

    def apply_AT(self, y_svec: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
        _need_cuda_f64(y_svec, "y_svec")
        x = torch.empty(self.m, dtype=torch.float64, device=y_svec.device)
        with torch.cuda.device(self.device):
            _check(load_library().hpsd_affine_apply_at(self._h, y_svec.data_ptr(), x.data_ptr(), _stream(stream)), "hpsd_affine_apply_at")
        return x

    def project_(self, a_x: torch.Tensor, a_y: torch.Tensor, z_x: torch.Tensor, z_y: torch.Tensor,
                 stream: Optional[torch.cuda.Stream] = None):
        for t, nm in ((a_x, "a_x"), (a_y, "a_y"), (z_x, "z_x"), (z_y, "z_y")):
            _need_cuda_f64(t, nm)
        with torch.cuda.device(self.device):
            _check(load_library().hpsd_affine_project(self._h, a_x.data_ptr(), a_y.data_ptr(), z_x.data_ptr(), z_y.data_ptr(),
                                                      _stream(stream)), "hpsd_affine_project")
        return z_x, z_y

    def destroy(self):
        if self._h:
            load_library().hpsd_affine_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def band_width() -> int:
    return int(load_library().hpsd_band_width())


def reduce_to_band(svec: torch.Tensor, n: int, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """hpsd_reduce_to_band: S2 alone.  Returns the band as an (n, 2b) complex tensor: row j holds column j of the
    band storage (element (i, j) of the band matrix at [j, i - j])."""
    _need_cuda_f64(svec, "svec")
    b = band_width()
    band = torch.empty((n, 2 * b), dtype=torch.complex128, device=svec.device)
    with torch.cuda.device(svec.device):
        _check(load_library().hpsd_reduce_to_band(n, svec.data_ptr(), band.data_ptr(), _stream(stream)), "hpsd_reduce_to_band")
    return band


def eigvalsh(svec: torch.Tensor, n: int, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    _need_cuda_f64(svec, "svec")
    lam = torch.empty(n, dtype=torch.float64, device=svec.device)
    with torch.cuda.device(svec.device):
        _check(load_library().hpsd_eigvalsh(n, svec.data_ptr(), lam.data_ptr(), _stream(stream)), "hpsd_eigvalsh")
    return lam


def profile_read() -> dict:
    """hpsd_profile_read: {stage name: (milliseconds, spans)} of the last call made with option profile=1."""
    lib = load_library()
    n = int(lib.hpsd_profile_stage_count())
    ms = (ctypes.c_double * n)()
    spans = (ctypes.c_int * n)()
    _check(lib.hpsd_profile_read(ms, spans, n), "hpsd_profile_read")
    return {lib.hpsd_profile_stage_name(i).decode(): (float(ms[i]), int(spans[i])) for i in range(n)}


def fp64_peak_probe(kind: int, iters: int, stream: Optional[torch.cuda.Stream] = None) -> float:
    """Enqueue the FP64 probe kernel; returns the flop count of the launch (time it with CUDA events)."""
    flops = ctypes.c_double(0.0)
    _check(load_library().hpsd_fp64_peak_probe(kind, iters, ctypes.byref(flops), _stream(stream)), "hpsd_fp64_peak_probe")
    return float(flops.value)
