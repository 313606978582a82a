"""ctypes loader for the CPU oracle (oracle/sh_oracle.c) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2510_05282_b200 (the CUDA path) and the CUDA
path imports nothing from here.  Arrays in and out are numpy float64; all outputs are AoS:
real [n][K], complex [n][K] complex128, spinor [n][2K][2] complex128 (up, down), K = (lmax+1)^2.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sh_oracle.c")
_LIB = os.path.join(_HERE, "libsh_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile sh_oracle.c with gcc (-O2, OpenMP, no fast-math) into oracle/libsh_oracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        for name in ("real", "complex", "spinor", "real_angular", "complex_angular", "spinor_angular"):
            f = getattr(lib, "sh_oracle_" + name)
            f.argtypes = [dp, ctypes.c_int64, ctypes.c_int, dp]
            f.restype = ctypes.c_int
        lib.sh_oracle_set_theta_mode.argtypes = [ctypes.c_int]
        lib.sh_oracle_set_threads.argtypes = [ctypes.c_int]
        lib.sh_oracle_threads_used.restype = ctypes.c_int
        lib.sh_oracle_max_imag_residue.restype = ctypes.c_double
        lib.sh_oracle_index_spinor.argtypes = [ctypes.c_int] * 3
        lib.sh_oracle_index_spinor.restype = ctypes.c_int
        ip = ctypes.POINTER(ctypes.c_int)
        lib.sh_oracle_projector_count.argtypes = [ctypes.c_int, ip]
        lib.sh_oracle_projector_count.restype = ctypes.c_int
        lib.sh_oracle_projectors.argtypes = [dp, ctypes.c_int64, ctypes.c_int, ip, dp, ctypes.c_int, ctypes.c_double, dp]
        lib.sh_oracle_projectors.restype = ctypes.c_int
        lib.sh_oracle_project.argtypes = [dp, ctypes.c_int64, ctypes.c_int, ip, dp, ctypes.c_int, ctypes.c_double, dp, ctypes.c_int, dp, dp]
        lib.sh_oracle_project.restype = ctypes.c_int
        _lib = lib
    return _lib


def _call(name: str, pts: np.ndarray, width: int, lmax: int, per_point: int) -> np.ndarray:
    lib = _load()
    a = np.ascontiguousarray(pts, dtype=np.float64)
    if a.ndim != 2 or a.shape[1] != width:
        raise ValueError(f"expected [n][{width}] array")
    n = a.shape[0]
    out = np.empty((n, per_point), dtype=np.float64)
    dp = ctypes.POINTER(ctypes.c_double)
    rc = getattr(lib, "sh_oracle_" + name)(a.ctypes.data_as(dp), n, int(lmax), out.ctypes.data_as(dp))
    if rc != 0:
        raise ValueError(f"sh_oracle_{name}: bad arguments (lmax={lmax}, n={n})")
    return out


def count(lmax: int) -> int:
    return (lmax + 1) ** 2


def real(xyz, lmax):
    """R_l^m at Cartesian points: [n][K] float64, k = l(l+1)+m."""
    return _call("real", xyz, 3, lmax, count(lmax))


def complex_(xyz, lmax):
    """Y_l^m at Cartesian points: [n][K] complex128."""
    return _call("complex", xyz, 3, lmax, 2 * count(lmax)).view(np.complex128)


def spinor(xyz, lmax):
    """Spin-1/2 spinor harmonics at Cartesian points: [n][2K][2] complex128 (up, down)."""
    return _call("spinor", xyz, 3, lmax, 8 * count(lmax)).view(np.complex128).reshape(len(xyz), 2 * count(lmax), 2)


def real_angular(theta_phi, lmax):
    return _call("real_angular", theta_phi, 2, lmax, count(lmax))


def complex_angular(theta_phi, lmax):
    return _call("complex_angular", theta_phi, 2, lmax, 2 * count(lmax)).view(np.complex128)


def spinor_angular(theta_phi, lmax):
    return _call("spinor_angular", theta_phi, 2, lmax, 8 * count(lmax)).view(np.complex128).reshape(
        len(theta_phi), 2 * count(lmax), 2
    )


def index_real(l: int, m: int) -> int:
    return l * (l + 1) + m


def index_spinor(l: int, twoj: int, twomj: int) -> int:
    return _load().sh_oracle_index_spinor(l, twoj, twomj)


def set_theta_mode(mode: int) -> None:
    """0 (default): Eq. 3 with the near-pole atan2 form; 1: literal acos everywhere."""
    _load().sh_oracle_set_theta_mode(int(mode))


def set_threads(t: int) -> None:
    _load().sh_oracle_set_threads(int(t))


def threads_used() -> int:
    return _load().sh_oracle_threads_used()


def max_imag_residue() -> float:
    return _load().sh_oracle_max_imag_residue()


def reset_imag_residue() -> None:
    _load().sh_oracle_reset_imag_residue()


# ---- fused projector consumer (definition in sh_oracle.c) ----
def _proj_args(xyz, proj_l, radial, dr):
    a = np.ascontiguousarray(xyz, dtype=np.float64)
    if a.ndim != 2 or a.shape[1] != 3:
        raise ValueError("expected [n][3] array")
    pl = np.ascontiguousarray(proj_l, dtype=np.int32)
    tab = np.ascontiguousarray(radial, dtype=np.float64)
    if tab.ndim != 2 or tab.shape[0] != len(pl):
        raise ValueError("radial must be [nproj][nr]")
    return a, pl, tab, float(dr)


def projector_count(proj_l) -> int:
    """ncols = sum_p (2 l_p + 1)."""
    pl = np.ascontiguousarray(proj_l, dtype=np.int32)
    return _load().sh_oracle_projector_count(len(pl), pl.ctypes.data_as(ctypes.POINTER(ctypes.c_int)))


def projectors(xyz, proj_l, radial, dr):
    """beta_{p,m}(r_i) = f_p(|r_i|) R_{l_p}^m(r_i/|r_i|): [n][ncols] float64 (columns channel-major, m ascending)."""
    a, pl, tab, dr = _proj_args(xyz, proj_l, radial, dr)
    ncols = projector_count(pl)
    out = np.empty((len(a), ncols), dtype=np.float64)
    dp, ip = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
    rc = _load().sh_oracle_projectors(a.ctypes.data_as(dp), len(a), len(pl), pl.ctypes.data_as(ip), tab.ctypes.data_as(dp),
                                      tab.shape[1], dr, out.ctypes.data_as(dp))
    if rc != 0:
        raise ValueError("sh_oracle_projectors: bad arguments")
    return out


def project(xyz, proj_l, radial, dr, w):
    """coeff[v][col] = sum_i w[v][i] beta_col(r_i) (plain long-double sum in point order) and the sums of |terms|:
    returns (coeff, abs_sum), both [nvec][ncols] float64."""
    a, pl, tab, dr = _proj_args(xyz, proj_l, radial, dr)
    ww = np.ascontiguousarray(w, dtype=np.float64)
    if ww.ndim != 2 or ww.shape[1] != len(a):
        raise ValueError("w must be [nvec][n]")
    ncols = projector_count(pl)
    coeff = np.empty((ww.shape[0], ncols), dtype=np.float64)
    abs_sum = np.empty_like(coeff)
    dp, ip = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
    rc = _load().sh_oracle_project(a.ctypes.data_as(dp), len(a), len(pl), pl.ctypes.data_as(ip), tab.ctypes.data_as(dp),
                                   tab.shape[1], dr, ww.ctypes.data_as(dp), ww.shape[0], coeff.ctypes.data_as(dp),
                                   abs_sum.ctypes.data_as(dp))
    if rc != 0:
        raise ValueError("sh_oracle_project: bad arguments")
    return coeff, abs_sum
