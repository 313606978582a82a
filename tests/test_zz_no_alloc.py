"""sh_project_static (include/shb200.h): sh_project for callers that cannot call cudaMalloc -- the per-CTA partial sums live in a
static device array inside the library (2 MiB) instead of a caller-provided workspace.

Collected LAST on purpose (the suite runs with `pytest -x`: a failure here must not hide another test).  The GPU tests compare the
new entry point with the existing path (sh_project with a workspace) on calls made back to back, so that what one call leaves in the
shared array is seen not to matter to the next; same kernels, same summation order, so the results are bit-identical, which is well
inside the tolerance the projector tests use (1e-12 sum_i |w_i beta_i|, tests/test_gpu_projector.py).  Every test passes alone in a
fresh process and after the other tests.
"""
import ctypes

import numpy as np
import pytest

TOL = 1e-12
SH_ERR_SCRATCH = -8


def _channels(lmax, per_l):
    from paper_2510_05282_b200 import inputs

    return inputs.projector_channels(lmax=lmax, per_l=per_l, cutoff=3.0, dr=0.01)


# ----------------------------------------------------------------------------- no GPU: the checks that precede every CUDA call
def test_static_entry_point_validates_before_any_cuda_call():
    import paper_2510_05282_b200 as sh
    from paper_2510_05282_b200 import build

    build.ensure_built()
    lib = sh.load()
    assert sh.project_static_bytes() == 2 << 20
    buf = np.zeros(64, dtype=np.float64)
    p = buf.ctypes.data
    ls = (ctypes.c_int * 3)(0, 1, 2)
    bad = (ctypes.c_int * 2)(0, 10)
    f = lib.sh_project_static
    assert f(p, -1, 3, ls, p, 8, 0.1, p, 1, p, None) == -2           # n < 0
    assert f(p, 4, 2, bad, p, 8, 0.1, p, 1, p, None) == -7           # l = 10
    assert f(p, 4, 3, ls, p, 1, 0.1, p, 1, p, None) == -7            # nr < 2
    assert f(p, 4, 3, ls, p, 8, 0.1, p, -1, p, None) == -7           # nvec < 0
    assert f(None, 4, 3, ls, p, 8, 0.1, p, 1, p, None) == -1         # xyz NULL
    assert f(p, 4, 3, ls, p, 8, 0.1, p, 0, None, None) == 0          # nvec = 0: nothing to do
    # beyond the static array: 8 vectors x 100 columns need 148 SMs x 4 CTAs x 800 doubles = 3.8 MB > 2 MiB (without a device the
    # library plans for 148 SMs), refused before anything is launched or looked up
    wide = (ctypes.c_int * 10)(*range(10))
    assert lib.sh_projector_count(10, wide) == 100
    assert lib.sh_project_workspace_bytes(100, 8) > sh.project_static_bytes()
    assert f(p, 4, 10, wide, p, 8, 0.1, p, 8, p, None) == SH_ERR_SCRATCH
    assert b"static scratch" in lib.sh_strerror(SH_ERR_SCRATCH)


# ----------------------------------------------------------------------------- GPU
@pytest.fixture(scope="module")
def sh():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2510_05282_b200 as pkg
    from paper_2510_05282_b200 import build

    build.ensure_built()
    pkg.load()
    return pkg


def _case(sh, pts, lmax, per_l, nvec, seed):
    """Device tensors of one projection problem and the existing path's result."""
    import torch

    from paper_2510_05282_b200 import inputs

    proj_l, tab, dr = _channels(lmax, per_l)
    x = torch.from_numpy(pts).cuda()
    t = torch.from_numpy(tab).cuda()
    w = torch.from_numpy(inputs.wave_weights(len(pts), nvec, seed=seed)).cuda()
    want = sh.sh_project(x, proj_l, t, dr, w)          # caller-provided workspace (allocated by the binding)
    beta = sh.sh_projectors(x, proj_l, t, dr, layout="soa")
    scale = (w.abs() @ beta.abs().T)                    # sum_i |w_i beta_i| per coefficient: the tolerance's scale
    torch.cuda.synchronize()
    return proj_l, tab, dr, x, t, w, want, scale


@pytest.mark.gpu
def test_static_scratch_matches_the_workspace_path_on_calls_in_a_row(sh):
    import torch

    from paper_2510_05282_b200 import inputs

    pts = inputs.config2_projector_grid()               # 113,102 points: every CTA of the persistent grids has several tiles
    cases = [
        _case(sh, pts, 3, 2, 4, seed=11),               # 32 columns, 4 vectors: ring kernel
        _case(sh, pts, 9, 1, 1, seed=12),               # 100 columns, 1 vector: segment kernel, wider rows than the call before
        _case(sh, pts[:1000], 9, 1, 3, seed=13),        # fewer CTAs than before: stale rows of the previous calls stay in the array
        _case(sh, pts, 3, 2, 4, seed=11),               # the first problem again, after the others
    ]
    outs = []
    for proj_l, tab, dr, x, t, w, want, scale in cases:  # back to back on one stream, no synchronization in between
        coeff = torch.full_like(want, float("nan"))
        sh.sh_project_static(x, proj_l, t, dr, w, coeff)
        outs.append(coeff)
    torch.cuda.synchronize()
    for k, ((_, _, _, _, _, _, want, scale), got) in enumerate(zip(cases, outs)):
        assert not torch.isnan(got).any(), k
        assert bool(((got - want).abs() <= TOL * scale).all()), (k, float((got - want).abs().max()))
        assert torch.equal(got, want), k                 # same kernels, same fixed summation order
    assert torch.equal(outs[0], outs[3])


@pytest.mark.gpu
def test_static_entry_point_allocates_nothing_and_refuses_what_does_not_fit(sh):
    import torch

    from paper_2510_05282_b200 import inputs

    pts = inputs.config2_projector_grid()[:50000]
    proj_l, tab, dr, x, t, w, want, scale = _case(sh, pts, 9, 1, 4, seed=21)   # 100 columns x 4 vectors: 1.9 MB of the 2 MiB
    coeff = torch.empty_like(want)
    sh.sh_project_static(x, proj_l, t, dr, w, coeff)    # first call on this device: symbol address looked up, kernels loaded
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        sh.sh_project_static(x, proj_l, t, dr, w, coeff)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0                                # no device memory was taken by the calls
    assert torch.equal(coeff, want)
    # 8 vectors x 100 columns need 3.8 MB on a 148-SM device: refused with SH_ERR_SCRATCH, nothing launched, coeff untouched
    w8 = torch.from_numpy(inputs.wave_weights(len(pts), 8, seed=22)).cuda()
    assert sh.project_workspace_bytes(100, 8) > sh.project_static_bytes()
    c8 = torch.full((8, 100), float("nan"), dtype=torch.float64, device="cuda")
    with pytest.raises(sh.ShError) as err:
        sh.sh_project_static(x, proj_l, t, dr, w8, c8)
    assert err.value.code == SH_ERR_SCRATCH
    torch.cuda.synchronize()
    assert torch.isnan(c8).all()
    # ... and the same request in two calls of four vectors fits: bit-identical to the existing path called the same way, and within the
    # projector tests' tolerance of the existing path's single eight-vector call (which sums in another fixed order)
    for v0 in (0, 4):
        sh.sh_project_static(x, proj_l, t, dr, w8[v0 : v0 + 4], c8[v0 : v0 + 4])
    torch.cuda.synchronize()
    for v0 in (0, 4):
        assert torch.equal(c8[v0 : v0 + 4], sh.sh_project(x, proj_l, t, dr, w8[v0 : v0 + 4].contiguous()))
    want8 = sh.sh_project(x, proj_l, t, dr, w8)
    scale8 = w8.abs() @ sh.sh_projectors(x, proj_l, t, dr, layout="soa").abs().T
    assert bool(((c8 - want8).abs() <= TOL * scale8).all())
    # the empty sum and the empty request
    e = torch.full((4, 100), float("nan"), dtype=torch.float64, device="cuda")
    sh.sh_project_static(x[:0], proj_l, t, dr, w[:, :0].contiguous(), e)
    torch.cuda.synchronize()
    assert bool((e == 0).all())


@pytest.mark.gpu
def test_static_entry_point_under_cuda_graph_capture(sh):
    """The motivating caller: the call captures into a CUDA graph (it allocates nothing and is asynchronous on its stream), and the
    replayed graph reproduces the existing path's result for new weights written into the captured buffer."""
    import torch

    from paper_2510_05282_b200 import inputs

    pts = inputs.config2_projector_grid()[:40000]
    proj_l, tab, dr, x, t, w, want, scale = _case(sh, pts, 3, 2, 2, seed=31)
    coeff = torch.empty_like(want)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        sh.sh_project_static(x, proj_l, t, dr, w, coeff)   # warm-up outside the capture (first-use set-up happens here)
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        sh.sh_project_static(x, proj_l, t, dr, w, coeff)
    w2 = torch.from_numpy(inputs.wave_weights(len(pts), 2, seed=32)).cuda()
    want2 = sh.sh_project(x, proj_l, t, dr, w2)
    w.copy_(w2)
    coeff.fill_(float("nan"))
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(coeff, want2)
