"""ctypes loader for libshb200_peaks.so (csrc/sh_peaks.cu): the ceilings microbenchmarks bench.py measures in the same run as
the kernels -- write-only fills in the library's store patterns and a DFMA chain.  Measurement code, not product path."""
from __future__ import annotations

import ctypes
import os

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libshb200_peaks.so")
_lib = None


def load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} not found: build it with `python -m paper_2510_05282_b200.build`")
        lib = ctypes.CDLL(LIB_PATH)
        vp, i64, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
        lib.shpeak_fill_flat.argtypes = [vp, i64, vp]
        lib.shpeak_fill_flat.restype = ci
        lib.shpeak_fill_bulk_tiles.argtypes = [vp, i64, ci, vp]
        lib.shpeak_fill_bulk_tiles.restype = ci
        lib.shpeak_fill_soa_planes.argtypes = [vp, i64, ci, ci, ci, vp]
        lib.shpeak_fill_soa_planes.restype = ci
        lib.shpeak_dfma.argtypes = [vp, i64, ci, vp]
        lib.shpeak_dfma.restype = i64
        _lib = lib
    return _lib


def _stream(t):
    import torch

    return torch.cuda.current_stream(t.device).cuda_stream


def fill_flat(out) -> None:
    """Every byte of the CUDA tensor `out` written once by 32-byte streaming stores."""
    if load().shpeak_fill_flat(out.data_ptr(), out.numel() * out.element_size(), _stream(out)) != 0:
        raise RuntimeError("shpeak_fill_flat failed")


def fill_bulk_tiles(out, tile_bytes: int) -> None:
    """`out` written as contiguous tiles of tile_bytes, one TMA bulk copy each (the AoS kernels' pattern)."""
    if load().shpeak_fill_bulk_tiles(out.data_ptr(), out.numel() * out.element_size(), int(tile_bytes), _stream(out)) != 0:
        raise RuntimeError("shpeak_fill_bulk_tiles failed")


def fill_soa_planes(out, row_doubles: int, planes: int) -> None:
    """`out` = float64 [k][row_total]: every {row_doubles x planes} box written by one TMA tensor store (the SoA kernels' pattern)."""
    k, row_total = out.shape
    if load().shpeak_fill_soa_planes(out.data_ptr(), row_total, k, int(row_doubles), int(planes), _stream(out)) != 0:
        raise RuntimeError("shpeak_fill_soa_planes failed")


def dfma(sink, iters: int, blocks: int) -> int:
    """Launches blocks x 256 threads of 8 independent DFMA chains, `iters` rounds; returns the DFMA lane-instructions executed."""
    r = int(load().shpeak_dfma(sink.data_ptr(), int(iters), int(blocks), _stream(sink)))
    if r < 0:
        raise RuntimeError("shpeak_dfma failed")
    return r
