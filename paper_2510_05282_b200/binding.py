"""Thin ctypes binding over libshb200.so (include/shb200.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels; PyTorch is used for device memory and streams.
There is no CPU fallback: if the shared library is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes
import math
import os

import numpy as np

SH_LAYOUT_AOS = 0
SH_LAYOUT_SOA = 1
SH_STORE_AUTO = 0 << 8
SH_STORE_DIRECT = 1 << 8
SH_STORE_BULK = 2 << 8

SH_COORDS_CARTESIAN = 0 << 16
SH_COORDS_NORMALIZED = 1 << 16
SH_COORDS_ANGULAR = 2 << 16

_COORDS = {"cartesian": SH_COORDS_CARTESIAN, "normalized": SH_COORDS_NORMALIZED, "angular": SH_COORDS_ANGULAR}
_LAYOUTS = {"aos": SH_LAYOUT_AOS, "soa": SH_LAYOUT_SOA, SH_LAYOUT_AOS: SH_LAYOUT_AOS, SH_LAYOUT_SOA: SH_LAYOUT_SOA}
_STORES = {"auto": SH_STORE_AUTO, "direct": SH_STORE_DIRECT, "bulk": SH_STORE_BULK}

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libshb200.so")
_lib = None


class ShError(RuntimeError):
    def __init__(self, code: int, where: str):
        lib = load()
        msg = lib.sh_strerror(code).decode()
        if code == -6:
            msg += ": " + lib.sh_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} (code {code})")
        self.code = code


def load() -> ctypes.CDLL:
    """Load libshb200.so; raises if it has not been built (python -m paper_2510_05282_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} not found: build it with `python -m paper_2510_05282_b200.build` (no CPU fallback exists)"
            )
        lib = ctypes.CDLL(LIB_PATH)
        vp, i64, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
        for name in ("sh_real_ext", "sh_complex_ext"):
            f = getattr(lib, name)
            f.argtypes = [vp, i64, ci, vp, ci, vp]
            f.restype = ci
        lib.sh_lmax_ext.restype = ci
        lib.sh_real_sum.argtypes = [vp, i64, ci, vp, ci, vp]
        lib.sh_real_sum.restype = ci
        for name in ("sh_real", "sh_complex", "sh_spinor", "sh_real_f32"):
            f = getattr(lib, name)
            f.argtypes = [vp, i64, ci, vp, ci, vp]
            f.restype = ci
            h = getattr(lib, name + "_host")
            h.argtypes = [vp, i64, ci, vp, ci]
            h.restype = ci
        for name in ("sh_real_count", "sh_complex_count", "sh_spinor_count"):
            getattr(lib, name).argtypes = [ci]
            getattr(lib, name).restype = i64
        lib.sh_index_real.argtypes = [ci, ci]
        lib.sh_index_real.restype = ci
        lib.sh_index_spinor.argtypes = [ci, ci, ci]
        lib.sh_index_spinor.restype = ci
        lib.sh_strerror.argtypes = [ci]
        lib.sh_strerror.restype = ctypes.c_char_p
        lib.sh_last_cuda_error.restype = ctypes.c_char_p
        lib.sh_kernel_launch_count.restype = i64
        lib.sh_host_release.restype = None
        ip = ctypes.POINTER(ci)
        lib.sh_projector_count.argtypes = [ci, ip]
        lib.sh_projector_count.restype = ci
        lib.sh_project_workspace_bytes.argtypes = [ci, ci]
        lib.sh_project_workspace_bytes.restype = i64
        lib.sh_projectors.argtypes = [vp, i64, ci, ip, vp, ci, ctypes.c_double, vp, ci, vp]
        lib.sh_projectors.restype = ci
        lib.sh_project.argtypes = [vp, i64, ci, ip, vp, ci, ctypes.c_double, vp, ci, vp, vp, i64, vp]
        lib.sh_project.restype = ci
        lib.sh_project_static.argtypes = [vp, i64, ci, ip, vp, ci, ctypes.c_double, vp, ci, vp, vp]
        lib.sh_project_static.restype = ci
        lib.sh_project_static_bytes.restype = i64
        _lib = lib
    return _lib


def layout_bits(layout, store="auto", coords="cartesian") -> int:
    return _LAYOUTS[layout] | _STORES[store] | _COORDS[coords]


def count(kind: str, lmax: int) -> int:
    """Scalars written per point."""
    return int(getattr(load(), f"sh_{_BASE_KIND.get(kind, kind)}_count")(lmax))


_BASE_KIND = {"real_f32": "real", "real_ext": "real", "complex_ext": "complex"}


def lmax_ext() -> int:
    """Largest lmax sh_real_ext / sh_complex_ext accept."""
    return int(load().sh_lmax_ext())


def index_real(l: int, m: int) -> int:
    return load().sh_index_real(l, m)


def index_spinor(l: int, twoj: int, twomj: int) -> int:
    return load().sh_index_spinor(l, twoj, twomj)


TUNE = {"prefetch_window_points": 0, "proj_aos_mode": 1, "soa_tma": 2, "project_form": 3, "proj_aos_split": 4, "soa_split": 5, "proj_aos_pairs": 6}


def set_tuning(knob, value: int) -> None:
    """sh_set_tuning: override a launch heuristic (include/shb200.h SH_TUNE_*); value 0 restores the default."""
    lib = load()
    lib.sh_set_tuning.argtypes = [ctypes.c_int, ctypes.c_int]
    lib.sh_set_tuning.restype = ctypes.c_int
    rc = lib.sh_set_tuning(TUNE[knob] if isinstance(knob, str) else int(knob), int(value))
    if rc != 0:
        raise ShError(rc, "sh_set_tuning")


def kernel_launch_count() -> int:
    return int(load().sh_kernel_launch_count())


def out_shape(kind: str, n: int, lmax: int, layout) -> tuple:
    """Shape of `out` in scalars: AoS [n][K*es], SoA [K][n*es] flattened per element as [K][n][es]."""
    k = (lmax + 1) ** 2
    es = {"real": 1, "real_f32": 1, "real_ext": 1, "complex": 2, "complex_ext": 2, "spinor": 4}[kind]
    ne = 2 * k if kind == "spinor" else k
    if _LAYOUTS[layout] == SH_LAYOUT_AOS:
        return (n, ne, es) if es > 1 else (n, ne)
    return (ne, n, es) if es > 1 else (ne, n)


def _current_stream(device) -> int:
    """cudaStream_t of torch's current stream on `device`, as an integer.  The raw query costs ~0.3 us against ~2.5 us for building a
    torch.cuda.Stream object -- a quarter of a launch-bound call (configs 1, 2); the public API is the fallback."""
    import torch

    raw = getattr(torch._C, "_cuda_getCurrentRawStream", None)
    if raw is not None:
        idx = device.index
        return int(raw(torch.cuda.current_device() if idx is None else idx))
    return int(torch.cuda.current_stream(device).cuda_stream)


def _device_call(kind: str, xyz, lmax: int, out, layout, store, stream, coords="cartesian"):
    import torch

    fn = getattr(load(), "sh_" + kind)
    want = torch.float32 if kind == "real_f32" else torch.float64
    width = 2 if coords == "angular" else 3
    if not (xyz.is_cuda and xyz.dtype == want and xyz.is_contiguous() and xyz.dim() == 2 and xyz.shape[1] == width):
        raise ValueError(f"xyz must be a contiguous CUDA tensor [n][{width}] of {want}")
    n = xyz.shape[0]
    shape = out_shape(kind, n, lmax, layout)
    if out is None:
        out = torch.empty(shape, dtype=want, device=xyz.device)
    elif not (out.is_cuda and out.dtype == want and out.is_contiguous() and out.numel() == math.prod(shape)):
        raise ValueError(f"out must be a contiguous CUDA tensor of {want} with {math.prod(shape)} elements")
    s = _current_stream(xyz.device) if stream is None else int(stream)
    args = (xyz.data_ptr(), n, int(lmax), out.data_ptr(), layout_bits(layout, store, coords), s)
    if xyz.device.index == torch.cuda.current_device():   # the usual case: no device switch (microseconds on launch-bound sizes)
        rc = fn(*args)
    else:
        with torch.cuda.device(xyz.device):
            rc = fn(*args)
    if rc != 0:
        raise ShError(rc, "sh_" + kind)
    return out


def sh_real(xyz, lmax, out=None, layout="soa", store="auto", stream=None, coords="cartesian"):
    """R_l^m (Eq. 6) for l <= lmax at CUDA tensor xyz [n][3] float64 -> AoS [n][K] or SoA [K][n].
    coords: "cartesian" (default), "normalized" (unit vectors, no normalization) or "angular" ([n][2] = theta, phi)."""
    return _device_call("real", xyz, lmax, out, layout, store, stream, coords)


def sh_complex(xyz, lmax, out=None, layout="soa", store="auto", stream=None, coords="cartesian"):
    """Y_l^m (Eq. 5) -> AoS [n][K][2] or SoA [K][n][2] float64 (re, im)."""
    return _device_call("complex", xyz, lmax, out, layout, store, stream, coords)


def sh_spinor(xyz, lmax, out=None, layout="soa", store="auto", stream=None, coords="cartesian"):
    """Spinor harmonics (Eq. 7) -> AoS [n][2K][4] or SoA [2K][n][4] float64 (up.re, up.im, down.re, down.im)."""
    return _device_call("spinor", xyz, lmax, out, layout, store, stream, coords)


def sh_real_f32(xyz, lmax, out=None, layout="soa", store="auto", stream=None, coords="cartesian"):
    """fp32 variant of sh_real (float32 in, float32 out)."""
    return _device_call("real_f32", xyz, lmax, out, layout, store, stream, coords)


def sh_real_sum(xyz, lmax, out=None, stream=None, coords="cartesian"):
    """out[i] = sum over l <= lmax, m of R_l^m(xyz_i): the accumulate-and-never-store protocol of the paper's Table I."""
    import torch

    width = 2 if coords == "angular" else 3
    if not (xyz.is_cuda and xyz.dtype == torch.float64 and xyz.is_contiguous() and xyz.dim() == 2 and xyz.shape[1] == width):
        raise ValueError(f"xyz must be a contiguous CUDA tensor [n][{width}] of float64")
    n = xyz.shape[0]
    if out is None:
        out = torch.empty(n, dtype=torch.float64, device=xyz.device)
    elif not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == n):
        raise ValueError(f"out must be a contiguous CUDA float64 tensor with {n} elements")
    s = _current_stream(xyz.device) if stream is None else int(stream)
    with torch.cuda.device(xyz.device):
        rc = load().sh_real_sum(xyz.data_ptr(), n, int(lmax), out.data_ptr(), _COORDS[coords], s)
    if rc != 0:
        raise ShError(rc, "sh_real_sum")
    return out


def sh_real_ext(xyz, lmax, out=None, layout="soa", store="auto", stream=None, coords="cartesian"):
    """R_l^m for l <= lmax <= 32: the explicit l <= 9 block plus the recurrence extension.  SoA only for lmax > 9."""
    return _device_call("real_ext", xyz, lmax, out, layout, store, stream, coords)


def sh_complex_ext(xyz, lmax, out=None, layout="soa", store="auto", stream=None, coords="cartesian"):
    """Y_l^m for l <= lmax <= 32 (see sh_real_ext)."""
    return _device_call("complex_ext", xyz, lmax, out, layout, store, stream, coords)


def host_call(kind: str, xyz, lmax: int, out=None, layout="soa", coords="cartesian"):
    """sh_*_host: HOST buffers in and out (numpy arrays or CPU torch tensors, ideally pinned).  `xyz` may be anything numpy
    can convert (it is copied if it is not a C-contiguous array of the right dtype); `out`, when given, is written in
    place and must therefore already be a C-contiguous array / CPU tensor of the right dtype and size."""
    fn = getattr(load(), f"sh_{kind}_host")
    dt = np.float32 if kind == "real_f32" else np.float64
    width = 2 if coords == "angular" else 3

    def is_tensor(a):
        return hasattr(a, "data_ptr")

    def check_tensor(a, what):
        import torch

        want = torch.float32 if kind == "real_f32" else torch.float64
        if a.is_cuda or a.dtype != want or not a.is_contiguous():
            raise ValueError(f"{what} must be a contiguous CPU tensor of {want}")

    if is_tensor(xyz):
        check_tensor(xyz, "xyz")
        if xyz.dim() != 2 or xyz.shape[1] != width:
            raise ValueError(f"xyz must be [n][{width}]")
        xp, xk = xyz.data_ptr(), xyz
    else:
        xk = np.ascontiguousarray(xyz, dtype=dt)
        if xk.ndim != 2 or xk.shape[1] != width:
            raise ValueError(f"xyz must be [n][{width}]")
        xp = xk.ctypes.data
    n = xk.shape[0]
    shape = out_shape(kind, n, lmax, layout)
    if out is None:
        out = np.empty(shape, dtype=dt)
    if is_tensor(out):
        check_tensor(out, "out")
        if out.numel() != math.prod(shape):
            raise ValueError(f"out must hold {math.prod(shape)} elements")
        op = out.data_ptr()
    else:
        if not (isinstance(out, np.ndarray) and out.dtype == dt and out.flags.c_contiguous and out.flags.writeable and out.size == math.prod(shape)):
            raise ValueError(f"out must be a writeable C-contiguous numpy array of {np.dtype(dt)} with {math.prod(shape)} elements")
        op = out.ctypes.data
    rc = fn(xp, n, int(lmax), op, _LAYOUTS[layout] | _COORDS[coords])
    if rc != 0:
        raise ShError(rc, f"sh_{kind}_host")
    return out


# ---- fused projector consumer (include/shb200.h "Fused projector consumer") ----
def _proj_l_array(proj_l):
    a = (ctypes.c_int * len(proj_l))(*[int(l) for l in proj_l])
    return a, len(proj_l)


def projector_count(proj_l) -> int:
    """ncols = sum_p (2 l_p + 1); raises if a channel is invalid."""
    a, k = _proj_l_array(proj_l)
    c = int(load().sh_projector_count(k, a))
    if c < 0:
        raise ShError(-7, "sh_projector_count")
    return c


def project_workspace_bytes(ncols: int, nvec: int) -> int:
    return int(load().sh_project_workspace_bytes(int(ncols), int(nvec)))


def _check_proj_inputs(xyz, radial, nproj):
    import torch

    if not (xyz.is_cuda and xyz.dtype == torch.float64 and xyz.is_contiguous() and xyz.dim() == 2 and xyz.shape[1] == 3):
        raise ValueError("xyz must be a contiguous CUDA tensor [n][3] of float64")
    if not (radial.is_cuda and radial.dtype == torch.float64 and radial.is_contiguous() and radial.dim() == 2 and radial.shape[0] == nproj):
        raise ValueError("radial must be a contiguous CUDA tensor [nproj][nr] of float64")


def sh_projectors(xyz, proj_l, radial, dr, out=None, layout="soa", stream=None):
    """beta_{p,m}(r_i) = f_p(|r_i|) R_{l_p}^m(r_i/|r_i|) -> AoS [n][ncols] or SoA [ncols][n]; radial [nproj][nr] at r_j = j dr."""
    import torch

    a, nproj = _proj_l_array(proj_l)
    _check_proj_inputs(xyz, radial, nproj)
    n, ncols = xyz.shape[0], projector_count(proj_l)
    shape = (n, ncols) if _LAYOUTS[layout] == SH_LAYOUT_AOS else (ncols, n)
    if out is None:
        out = torch.empty(shape, dtype=torch.float64, device=xyz.device)
    elif not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == n * ncols):
        raise ValueError(f"out must be a contiguous CUDA float64 tensor with {n * ncols} elements")
    s = _current_stream(xyz.device) if stream is None else int(stream)
    with torch.cuda.device(xyz.device):
        rc = load().sh_projectors(xyz.data_ptr(), n, nproj, a, radial.data_ptr(), radial.shape[1], float(dr), out.data_ptr(), _LAYOUTS[layout], s)
    if rc != 0:
        raise ShError(rc, "sh_projectors")
    return out


def sh_project(xyz, proj_l, radial, dr, w, coeff=None, workspace=None, stream=None):
    """coeff[v][col] = sum_i w[v][i] beta_col(r_i); w [nvec][n] CUDA float64 -> coeff [nvec][ncols].  `workspace` (a CUDA
    uint8 tensor of at least project_workspace_bytes(ncols, nvec) bytes) is allocated with PyTorch when not given."""
    import torch

    a, nproj = _proj_l_array(proj_l)
    _check_proj_inputs(xyz, radial, nproj)
    n, ncols = xyz.shape[0], projector_count(proj_l)
    if not (w.is_cuda and w.dtype == torch.float64 and w.is_contiguous() and w.dim() == 2 and w.shape[1] == n):
        raise ValueError("w must be a contiguous CUDA tensor [nvec][n] of float64")
    nvec = w.shape[0]
    if coeff is None:
        coeff = torch.empty((nvec, ncols), dtype=torch.float64, device=xyz.device)
    elif not (coeff.is_cuda and coeff.dtype == torch.float64 and coeff.is_contiguous() and coeff.numel() == nvec * ncols):
        raise ValueError(f"coeff must be a contiguous CUDA float64 tensor with {nvec * ncols} elements")
    need = project_workspace_bytes(ncols, nvec)
    if workspace is None:
        workspace = torch.empty(max(need, 8), dtype=torch.uint8, device=xyz.device)
    s = _current_stream(xyz.device) if stream is None else int(stream)
    with torch.cuda.device(xyz.device):
        rc = load().sh_project(xyz.data_ptr(), n, nproj, a, radial.data_ptr(), radial.shape[1], float(dr), w.data_ptr(), nvec,
                               coeff.data_ptr(), workspace.data_ptr(), workspace.numel() * workspace.element_size(), s)
    if rc != 0:
        raise ShError(rc, "sh_project")
    return coeff


def project_static_bytes() -> int:
    """Size of the static scratch array sh_project_static works in (2 MiB)."""
    return int(load().sh_project_static_bytes())


def sh_project_static(xyz, proj_l, radial, dr, w, coeff, stream=None):
    """sh_project without any allocation (include/shb200.h "sh_project_static"): the per-CTA partial sums live in a static device
    array inside the library, so `coeff` [nvec][ncols] must be given and nothing is allocated here either.  Raises ShError with
    code -8 (SH_ERR_SCRATCH) when the request needs more than project_static_bytes().  Calls that overlap on the GPU race."""
    import torch

    a, nproj = _proj_l_array(proj_l)
    _check_proj_inputs(xyz, radial, nproj)
    n, ncols = xyz.shape[0], projector_count(proj_l)
    if not (w.is_cuda and w.dtype == torch.float64 and w.is_contiguous() and w.dim() == 2 and w.shape[1] == n):
        raise ValueError("w must be a contiguous CUDA tensor [nvec][n] of float64")
    nvec = w.shape[0]
    if not (coeff.is_cuda and coeff.dtype == torch.float64 and coeff.is_contiguous() and coeff.numel() == nvec * ncols):
        raise ValueError(f"coeff must be a contiguous CUDA float64 tensor with {nvec * ncols} elements")
    s = _current_stream(xyz.device) if stream is None else int(stream)
    with torch.cuda.device(xyz.device):
        rc = load().sh_project_static(xyz.data_ptr(), n, nproj, a, radial.data_ptr(), radial.shape[1], float(dr), w.data_ptr(), nvec,
                                      coeff.data_ptr(), s)
    if rc != 0:
        raise ShError(rc, "sh_project_static")
    return coeff
