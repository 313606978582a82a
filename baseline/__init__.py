"""ctypes loader for baseline/sh_cpu_method.cpp: the paper's method (generated factorized formulas, fp64) on the host
cores.  A CHECK and a timed BASELINE, never a fallback: only tests/ and bench.py's `cpu_method` leg import this package;
paper_2510_05282_b200 (the product) never does, and nothing here imports oracle/.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sh_cpu_method.cpp")
_GEN = os.path.join(_HERE, "..", "paper_2510_05282_b200", "csrc", "sh_generated.cuh")
_LIB = os.path.join(_HERE, "libsh_cpu_method.so")
_lib = None


def build(force: bool = False) -> str:
    """g++ -O3 (no fast-math), OpenMP, function multiversioning for AVX2+FMA / AVX-512 resolved at load time, so the
    library built on one machine runs on another."""
    deps = [_SRC, _GEN]
    if force or not os.path.exists(_LIB) or any(os.path.getmtime(_LIB) < os.path.getmtime(d) for d in deps):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O3", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-Wall", "-Wno-psabi", "-x", "c++", _SRC,
                               "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        lib.shcpu_real.argtypes = [dp, ctypes.c_int64, ctypes.c_int, dp, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        lib.shcpu_real.restype = ctypes.c_int
        lib.shcpu_real_accumulate_l9.argtypes = [dp, ctypes.c_int64, ctypes.c_int, ctypes.c_int]
        lib.shcpu_real_accumulate_l9.restype = ctypes.c_double
        lib.shcpu_set_threads.argtypes = [ctypes.c_int]
        lib.shcpu_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def real(xyz, lmax: int, layout: str = "aos", normalized: bool = False, form: str = "factorized", out=None) -> np.ndarray:
    """R_l^m, l <= lmax, at xyz [n][3] float64 -> AoS [n][K] or SoA [K][n]."""
    lib = _load()
    a = np.ascontiguousarray(xyz, dtype=np.float64)
    if a.ndim != 2 or a.shape[1] != 3:
        raise ValueError("expected [n][3] array")
    n, k = a.shape[0], (lmax + 1) ** 2
    shape = (n, k) if layout == "aos" else (k, n)
    if out is None:
        out = np.empty(shape, dtype=np.float64)
    elif not (out.dtype == np.float64 and out.flags.c_contiguous and out.size == n * k):
        raise ValueError("out must be a C-contiguous float64 array of n*K elements")
    dp = ctypes.POINTER(ctypes.c_double)
    rc = lib.shcpu_real(a.ctypes.data_as(dp), n, int(lmax), out.ctypes.data_as(dp), int(layout == "soa"), int(normalized),
                        {"factorized": 0, "horner": 1}[form])
    if rc != 0:
        raise ValueError(f"shcpu_real: bad arguments (lmax={lmax}, n={n})")
    return out


def accumulate_l9(xyz, normalized: bool = False, form: str = "factorized") -> float:
    """Sum of all lmax = 9 harmonics over the batch, nothing stored (the paper's timing loop)."""
    a = np.ascontiguousarray(xyz, dtype=np.float64)
    return float(_load().shcpu_real_accumulate_l9(a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), a.shape[0], int(normalized),
                                                  {"factorized": 0, "horner": 1}[form]))


def set_threads(t: int) -> None:
    """t <= 0: all cores."""
    _load().shcpu_set_threads(int(t))


def threads() -> int:
    return int(_load().shcpu_threads())
