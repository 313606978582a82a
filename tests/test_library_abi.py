"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/shb200.h declares,
and validates arguments before touching the GPU.  No kernel is launched here."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2510_05282_b200 import build, binding

    build.build()
    return binding.load()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "shb200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sh_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = declared_functions()
    assert len(names) >= 16 and "sh_real" in names and "sh_spinor_host" in names
    for name in names:
        assert hasattr(lib, name), name


def test_counts_and_indices(lib):
    for lmax in range(10):
        k = (lmax + 1) ** 2
        assert lib.sh_real_count(lmax) == k and lib.sh_complex_count(lmax) == 2 * k and lib.sh_spinor_count(lmax) == 8 * k
    # real / complex counts and indices reach l = 32, the range of sh_real_ext / sh_complex_ext; spinors stop at 9
    assert lib.sh_lmax_ext() == 32
    assert lib.sh_real_count(32) == 1089 and lib.sh_complex_count(32) == 2178
    assert lib.sh_real_count(33) == -1 and lib.sh_spinor_count(10) == -1 and lib.sh_spinor_count(-1) == -1
    assert [lib.sh_index_real(l, m) for l in range(33) for m in range(-l, l + 1)] == list(range(1089))
    assert lib.sh_index_real(3, 4) == -1 and lib.sh_index_real(33, 0) == -1
    seen = []
    for l in range(10):
        for twoj in (2 * l - 1, 2 * l + 1):
            if twoj < 1:
                continue
            seen += [lib.sh_index_spinor(l, twoj, tm) for tm in range(-twoj, twoj + 1, 2)]
    assert seen == list(range(200))
    assert lib.sh_index_spinor(0, -1, 1) == -1 and lib.sh_index_spinor(2, 5, 4) == -1 and lib.sh_index_spinor(2, 5, 7) == -1


def test_argument_validation_without_gpu(lib):
    """Errors are returned before any CUDA call (P: boundary contract in include/shb200.h)."""
    buf = np.zeros(64, dtype=np.float64)
    p = buf.ctypes.data
    for fn in (lib.sh_real, lib.sh_complex, lib.sh_spinor, lib.sh_real_f32):
        assert fn(p, -1, 3, p, 0, None) == -2            # SH_ERR_COUNT
        assert fn(p, 4, 10, p, 0, None) == -3            # SH_ERR_LMAX
        assert fn(p, 4, -1, p, 1, None) == -3
        assert fn(p, 4, 3, p, 2, None) == -4             # SH_ERR_LAYOUT
        assert fn(p, 4, 3, p, 0 | (3 << 8), None) == -4
        assert fn(p, 4, 3, p, 0 | (3 << 16), None) == -4  # unknown front end
        assert fn(p, 4, 3, p, 1 | (1 << 18), None) == -4
        assert fn(None, 4, 3, p, 0, None) == -1          # SH_ERR_NULL
        assert fn(p, 4, 3, None, 1, None) == -1
        assert fn(None, 0, 3, None, 0, None) == 0        # n = 0: successful no-op
    assert lib.sh_real(p, 4, 3, p + 4, 0, None) == -5    # SH_ERR_ALIGNMENT
    for fn in (lib.sh_real_ext, lib.sh_complex_ext):
        assert fn(p, -1, 20, p, 1, None) == -2 and fn(p, 4, 33, p, 1, None) == -3 and fn(p, 4, -1, p, 1, None) == -3
        assert fn(p, 4, 10, p, 0, None) == -4            # AoS is not offered above lmax = 9
        assert fn(p, 4, 20, p, 1 | (2 << 8), None) == -4  # nor the bulk store path
        assert fn(None, 4, 20, p, 1, None) == -1 and fn(None, 0, 20, None, 1, None) == 0
        assert fn(p, 4, 20, p + 4, 1, None) == -5
    # sh_real_sum: `coords` is one SH_COORDS_* value, no layout bits
    f = lib.sh_real_sum
    assert f(p, -1, 3, p, 0, None) == -2 and f(p, 4, 10, p, 0, None) == -3 and f(p, 4, -1, p, 0, None) == -3
    assert f(p, 4, 3, p, 1, None) == -4 and f(p, 4, 3, p, 3 << 16, None) == -4          # a layout bit, an unknown front end
    assert f(None, 4, 3, p, 0, None) == -1 and f(p, 4, 3, None, 1 << 16, None) == -1
    assert f(p, 4, 3, p + 4, 2 << 16, None) == -5 and f(None, 0, 3, None, 0, None) == 0
    for fn in (lib.sh_real_host, lib.sh_complex_host, lib.sh_spinor_host, lib.sh_real_f32_host):
        assert fn(p, -1, 3, p, 0) == -2 and fn(p, 1, 11, p, 0) == -3 and fn(None, 0, 3, None, 1) == 0
    # fused projector consumer: every argument is checked on the host
    ip = ctypes.POINTER(ctypes.c_int)
    ls = (ctypes.c_int * 3)(0, 1, 2)
    bad = (ctypes.c_int * 2)(0, 10)
    assert lib.sh_projector_count(3, ls) == 9 and lib.sh_projector_count(0, None) == 0
    assert lib.sh_projector_count(2, bad) == -1 and lib.sh_projector_count(33, ls) == -1 and lib.sh_projector_count(-1, ls) == -1
    assert lib.sh_project_workspace_bytes(-1, 1) == -1 and lib.sh_project_workspace_bytes(9, -1) == -1
    assert lib.sh_projectors(p, -1, 3, ls, p, 8, 0.1, p, 1, None) == -2          # n < 0
    assert lib.sh_projectors(p, 4, 2, bad, p, 8, 0.1, p, 1, None) == -7          # l = 10
    assert lib.sh_projectors(p, 4, 3, ls, p, 1, 0.1, p, 1, None) == -7           # nr < 2
    assert lib.sh_projectors(p, 4, 3, ls, p, 8, 0.0, p, 1, None) == -7           # dr <= 0
    assert lib.sh_projectors(p, 4, 3, ls, p, 8, float("nan"), p, 1, None) == -7
    assert lib.sh_projectors(None, 4, 3, ls, p, 8, 0.1, p, 1, None) == -1
    assert lib.sh_projectors(p, 4, 3, ls, None, 8, 0.1, p, 1, None) == -1
    assert lib.sh_projectors(p, 4, 3, ls, p, 8, 0.1, None, 1, None) == -1
    assert lib.sh_projectors(p, 4, 3, ls, p, 8, 0.1, p, 2, None) == -4           # layout
    assert lib.sh_projectors(p, 4, 3, ls, p, 8, 0.1, p, 1 | (1 << 16), None) == -4  # Cartesian points only
    assert lib.sh_projectors(p, 4, 3, ls, p, 8, 0.1, p + 4, 1, None) == -5
    assert lib.sh_projectors(None, 0, 3, ls, None, 8, 0.1, None, 0, None) == 0   # n = 0
    assert lib.sh_project(p, -1, 3, ls, p, 8, 0.1, p, 1, p, p, 1 << 30, None) == -2
    assert lib.sh_project(p, 4, 3, ls, p, 8, 0.1, p, -1, p, p, 1 << 30, None) == -7
    assert lib.sh_project(p, 4, 3, ls, p, 8, 0.1, None, 1, p, p, 1 << 30, None) == -1
    assert lib.sh_project(p, 4, 3, ls, p, 8, 0.1, p, 1, None, p, 1 << 30, None) == -1
    assert lib.sh_project(p, 4, 3, ls, p, 8, 0.1, p, 0, None, None, 0, None) == 0  # nvec = 0
    for code in range(-7, 1):
        assert len(lib.sh_strerror(code)) > 1
    assert lib.sh_strerror(-99) == b"unknown error code"


def test_binding_fails_loudly_without_library(monkeypatch, tmp_path):
    from paper_2510_05282_b200 import binding

    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "missing.so"))
    with pytest.raises(FileNotFoundError):
        binding.load()


def test_generator_output_is_current():
    """csrc/sh_generated.cuh is exactly what the generator emits (committed copy is not stale)."""
    from paper_2510_05282_b200.gen import generate

    generate.self_check()
    generate.self_check_recurrence()
    path = os.path.join(ROOT, "paper_2510_05282_b200", "csrc", "sh_generated.cuh")
    assert open(path).read() == generate.emit()


def test_peaks_library_exports_its_entry_points():
    """csrc/sh_peaks.cu -> libshb200_peaks.so: the ceilings microbenchmarks bench.py measures in the same run (no launch here)."""
    from paper_2510_05282_b200 import build, peaks

    build.build_peaks()
    lib = peaks.load()
    for name in ("shpeak_fill_flat", "shpeak_fill_bulk_tiles", "shpeak_fill_soa_planes", "shpeak_dfma"):
        assert hasattr(lib, name), name
    assert lib.shpeak_fill_flat(None, 64, None) == -1 and lib.shpeak_fill_bulk_tiles(None, 64, 16, None) == -1
    assert lib.shpeak_fill_soa_planes(None, 64, 4, 32, 4, None) == -1 and lib.shpeak_dfma(None, 1, 1, None) == -1


def test_host_call_validates_buffers_before_the_library_sees_them(lib):
    """binding.host_call: a wrong dtype, a strided or too-small `out` must raise instead of letting sh_*_host write out of bounds."""
    import torch

    import paper_2510_05282_b200 as sh

    pts = np.zeros((5, 3))
    with pytest.raises(ValueError):
        sh.host_call("real", pts, 3, out=np.empty((5, 16), dtype=np.float32))
    with pytest.raises(ValueError):
        sh.host_call("real", pts, 3, out=np.empty((5, 15)))
    with pytest.raises(ValueError):
        sh.host_call("real", pts, 3, out=np.empty((5, 32))[:, ::2])
    with pytest.raises(ValueError):
        sh.host_call("real", np.zeros((5, 2)), 3)
    with pytest.raises(ValueError):
        sh.host_call("real", torch.zeros((5, 3), dtype=torch.float32), 3)
    with pytest.raises(ValueError):
        sh.host_call("real", torch.zeros((5, 3), dtype=torch.float64), 3, out=torch.zeros((5, 16), dtype=torch.float64)[:, ::2])
    with pytest.raises(ValueError):
        sh.host_call("real_f32", torch.zeros((5, 3), dtype=torch.float32), 3, out=torch.zeros(5 * 16 - 1, dtype=torch.float32))
