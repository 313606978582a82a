"""paper_2510_05282_b200: batched real / complex / spinor spherical harmonics (l <= 9) on one B200.

The product is the C-ABI library libshb200.so (include/shb200.h, csrc/*.cu); this package holds the
build step, the build-time formula generator, a thin ctypes binding and the seeded workload generators.
"""
from .binding import (  # noqa: F401
    SH_LAYOUT_AOS,
    SH_LAYOUT_SOA,
    ShError,
    count,
    host_call,
    index_real,
    index_spinor,
    kernel_launch_count,
    load,
    out_shape,
    project_workspace_bytes,
    projector_count,
    set_tuning,
    lmax_ext,
    sh_complex,
    sh_complex_ext,
    sh_project,
    sh_project_static,
    project_static_bytes,
    sh_projectors,
    sh_real,
    sh_real_ext,
    sh_real_f32,
    sh_real_sum,
    sh_spinor,
)
