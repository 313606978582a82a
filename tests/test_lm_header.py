"""include/shb200_lm.cuh, the header-only per-(l, m) interface (the paper's own API shape), compiled as plain C++
with g++ and compared with the oracle at random unit vectors.  No GPU."""
import ctypes
import os
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def harness(tmp_path_factory):
    so = str(tmp_path_factory.mktemp("lm") / "liblm_harness.so")
    subprocess.check_call(["g++", "-std=c++17", "-O1", "-shared", "-fPIC", "-o", so, os.path.join(ROOT, "tests", "lm_harness.cpp")])
    lib = ctypes.CDLL(so)
    lib.lm_eval.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
    lib.lm_eval.restype = None
    lib.lm_real_7_m3_f32.argtypes = [ctypes.c_float] * 3
    lib.lm_real_7_m3_f32.restype = ctypes.c_float
    return lib


def test_every_lm_matches_the_oracle(harness):
    import oracle

    oracle.build()
    rng = np.random.default_rng(77)
    g = rng.standard_normal((2000, 3))
    g[0] = (0.0, 0.0, 1.0)      # poles and axis points
    g[1] = (0.0, 0.0, -1.0)
    g[2] = (1.0, 0.0, 0.0)
    g[3] = (0.0, -1.0, 0.0)
    u = np.ascontiguousarray(g / np.linalg.norm(g, axis=1)[:, None])
    real = np.empty((len(u), 100))
    cplx = np.empty((len(u), 100, 2))
    harness.lm_eval(u.ctypes.data, len(u), real.ctypes.data, cplx.ctypes.data)
    assert np.abs(real - oracle.real(u, 9)).max() <= 3e-14
    want_c = oracle.complex_(u, 9).view(np.float64).reshape(len(u), 100, 2)
    assert np.abs(cplx - want_c).max() <= 3e-14


def test_worked_example_in_fp32(harness):
    """R_7^{-3}, the paper's worked example (Eq. 11-15), through the float instantiation."""
    import oracle

    oracle.build()
    v = np.array([[0.3, -0.5, 0.2]])
    v /= np.linalg.norm(v)
    v32 = v.astype(np.float32)
    got = harness.lm_real_7_m3_f32(*[float(c) for c in v32[0]])
    want = oracle.real(v32.astype(np.float64) / np.linalg.norm(v32.astype(np.float64)), 9)[0, 7 * 8 - 3]
    assert abs(got - want) <= 1e-5
