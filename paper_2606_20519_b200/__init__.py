"""B200-native Hermitian PSD-cone projection (hot path of arxiv/paper_2606_20519).

Thin Python binding over the C-ABI library libhpsd.so (include/hpsd.h).  Every step of
the path runs in the library's CUDA kernels; this package only marshals arguments.
PyTorch is used for device memory and streams only.  There is no CPU fallback: if the
CUDA extension is missing or no GPU is present, calls raise.
"""
from .binding import (  # noqa: F401
    HpsdError,
    admm_step_,
    eigvalsh,
    Plan,
    Affine,
    project_approx,
    project_static_,
    svec_convert,
    reduce_to_band,
    band_width,
    fp64_peak_probe,
    last_launch_count,
    lib_path,
    load_library,
    pack,
    project,
    project_,
    project_host,
    project_ws,
    profile_read,
    release,
    set_option,
    svec_len,
    tridiagonalize,
    unpack,
    version,
    workspace_size,
    EXPORTS,
)
from .sharding import assign_blocks, project_sharded  # noqa: F401
