"""Build step: run the generator, then compile csrc/*.cu for sm_100a (one nvcc per translation unit, in parallel) and
link them into libshb200.so (in-tree).

    python -m paper_2510_05282_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libshb200.so")
PEAKS_LIB = os.path.join(HERE, "libshb200_peaks.so")   # ceilings microbenchmarks (csrc/sh_peaks.cu): bench.py only, never linked into LIB
# one harmonic kind per unit (they compile in parallel), the l > 9 extension, the fused projector consumer, shared host state
SOURCES = ["sh_real.cu", "sh_complex.cu", "sh_spinor.cu", "sh_real_f32.cu", "sh_ext.cu", "sh_projector.cu", "sh_abi.cu"]
HEADERS = ["sh_core.cuh", "sh_store.cuh", "sh_generated.cuh"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17", "--expt-relaxed-constexpr",
    "-Xcompiler", "-fPIC",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def generate() -> str:
    from .gen import generate as g

    return g.main(["generate.py", os.path.join(CSRC, "sh_generated.cuh")])


def build(force: bool = False, verbose: bool = False, extra_flags: tuple = ()) -> str:
    """Objects go to csrc/build/ (git-ignored); a unit is recompiled when it, a header or the flags changed."""
    generate()
    common = [os.path.join(HERE, "..", "include", "shb200.h")] + [os.path.join(CSRC, h) for h in HEADERS]
    flags = NVCC_FLAGS + list(extra_flags) + (["-Xptxas", "-v"] if verbose else [])
    objdir = os.path.join(CSRC, "build")
    os.makedirs(objdir, exist_ok=True)
    stamp = os.path.join(objdir, "flags.txt")
    if not os.path.exists(stamp) or open(stamp).read() != " ".join(flags):
        force = True
    jobs = []
    for s in SOURCES:
        src, obj = os.path.join(CSRC, s), os.path.join(objdir, s[:-3] + ".o")
        if force or not os.path.exists(obj) or any(os.path.getmtime(obj) < os.path.getmtime(d) for d in [src] + common):
            jobs.append((s, obj, subprocess.Popen([_nvcc()] + flags + ["-c", src, "-o", obj])))
    failed = [s for s, _, proc in jobs if proc.wait() != 0]
    if failed:
        for s, obj, _ in jobs:
            if s in failed and os.path.exists(obj):
                os.remove(obj)
        raise RuntimeError("nvcc failed for " + ", ".join(failed))
    with open(stamp, "w") as f:
        f.write(" ".join(flags))
    build_peaks()
    objs = [os.path.join(objdir, s[:-3] + ".o") for s in SOURCES]
    if not jobs and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(o) for o in objs):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call([_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs)
    os.replace(tmp, LIB)
    return LIB


def build_peaks(force: bool = False) -> str:
    """csrc/sh_peaks.cu -> libshb200_peaks.so: the write-only fill and DFMA ceilings bench.py measures in the same run."""
    src = os.path.join(CSRC, "sh_peaks.cu")
    if force or not os.path.exists(PEAKS_LIB) or os.path.getmtime(PEAKS_LIB) < os.path.getmtime(src):
        tmp = PEAKS_LIB + f".tmp{os.getpid()}"
        subprocess.check_call([_nvcc()] + NVCC_FLAGS + ["-shared", "-o", tmp, src])
        os.replace(tmp, PEAKS_LIB)
    return PEAKS_LIB


def ensure_built() -> str:
    """Compile only if libshb200.so is absent (a fresh checkout on a box that has nvcc).  Never a fallback: the result is
    the same CUDA library, and binding.load() still raises if it cannot be produced."""
    if not os.path.exists(PEAKS_LIB):
        build_peaks()
    return LIB if os.path.exists(LIB) else build(force=True)


if __name__ == "__main__":
    # extra nvcc -D flags pass through
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, extra_flags=tuple(a for a in sys.argv[1:] if a.startswith("-D"))))
