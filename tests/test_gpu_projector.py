"""GPU parity of the fused projector consumer (sh_projectors / sh_project, include/shb200.h; SURVEY.md section 8(f2);
PAPER.md lines 14, 20) against the CPU oracle on the same seeded inputs.

Tolerances:
  sh_projectors: |beta_gpu - beta_oracle| <= 1e-12 max(1, max |radial|)  -- north_star's fp64 bound, scaled by the table
  sh_project:    |c_gpu - c_oracle| <= 1e-12 sum_i |w_i beta_i| -- the same relative bound on the summands; the GPU adds in
                 a different (fixed) order than the oracle's plain point-order long-double sum.
Run on the B200 box: python -m pytest tests -m gpu.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-12


@pytest.fixture(scope="module")
def sh():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2510_05282_b200 as pkg
    from paper_2510_05282_b200 import build

    build.ensure_built()   # compiles only if the in-tree library is absent
    pkg.load()
    return pkg


def gpu_projectors(sh, pts, proj_l, tab, dr, layout, misalign=0):
    import torch

    x = torch.from_numpy(np.ascontiguousarray(pts)).cuda()
    t = torch.from_numpy(np.ascontiguousarray(tab)).cuda()
    n, ncols = len(pts), sh.projector_count(proj_l) if len(proj_l) else 0
    backing = torch.full((n * ncols + 8,), float("nan"), dtype=torch.float64, device="cuda")
    out = backing[misalign : misalign + n * ncols]
    sh.sh_projectors(x, proj_l, t, dr, out=out, layout=layout)
    torch.cuda.synchronize()
    assert torch.isnan(backing[:misalign]).all() and torch.isnan(backing[misalign + n * ncols :]).all()
    res = out.cpu().numpy()
    return res.reshape(n, ncols) if layout == "aos" else np.ascontiguousarray(res.reshape(ncols, n).T)


def gpu_project(sh, pts, proj_l, tab, dr, w):
    import torch

    x = torch.from_numpy(np.ascontiguousarray(pts)).cuda()
    t = torch.from_numpy(np.ascontiguousarray(tab)).cuda()
    ww = torch.from_numpy(np.ascontiguousarray(w)).cuda()
    c = sh.sh_project(x, proj_l, t, dr, ww)
    torch.cuda.synchronize()
    return c.cpu().numpy()


def check_project(got, coeff, abs_sum):
    bound = TOL * abs_sum + 1e-300
    bad = np.abs(got - coeff) > bound
    assert not bad.any(), (np.abs(got - coeff)[bad].max(), abs_sum[bad].min())
    # report how far inside the bound the run is
    return float((np.abs(got - coeff) / (abs_sum + 1e-300)).max())


@pytest.fixture(scope="module")
def grid2():
    from paper_2510_05282_b200 import inputs

    return inputs.config2_projector_grid()   # 113,102 lattice points within 3 bohr of an atom at a sub-grid offset


@pytest.mark.parametrize("layout", ["soa", "aos"])
def test_projector_grid_values(sh, oracle_mod, grid2, layout):
    from paper_2510_05282_b200 import inputs

    proj_l, tab, dr = inputs.projector_channels(lmax=3, per_l=2)   # 8 channels, 32 columns, cutoff 3.0
    got = gpu_projectors(sh, grid2, proj_l, tab, dr, layout)
    want = oracle_mod.projectors(grid2, proj_l, tab, dr)
    assert got.shape == want.shape == (len(grid2), 32)
    assert np.abs(got - want).max() <= TOL * max(1.0, np.abs(tab).max())


@pytest.mark.parametrize("nvec", [1, 2, 3, 4, 6, 8, 11])   # one vector: segment kernel; 2-4 and 5-8: ring kernel; 11 = 8 + 3 in two passes
def test_projector_grid_projection(sh, oracle_mod, grid2, nvec):
    from paper_2510_05282_b200 import inputs

    proj_l, tab, dr = inputs.projector_channels(lmax=3, per_l=2)
    w = inputs.wave_weights(len(grid2), nvec)
    got = gpu_project(sh, grid2, proj_l, tab, dr, w)
    coeff, abs_sum = oracle_mod.project(grid2, proj_l, tab, dr, w)
    assert got.shape == (nvec, 32)
    check_project(got, coeff, abs_sum)
    # reproducible: the summation order is fixed
    assert np.array_equal(got, gpu_project(sh, grid2, proj_l, tab, dr, w))


@pytest.mark.parametrize("lmax", range(10))
def test_every_lmax_unsorted_channels_and_ragged_sizes(sh, oracle_mod, lmax):
    rng = np.random.default_rng(100 + lmax)
    # unsorted channel list with repeats that reaches lmax and skips some l-blocks
    proj_l = [lmax] + [int(v) for v in rng.integers(0, lmax + 1, 4)] + [lmax // 2]
    nr, dr = 57, 0.05
    tab = rng.standard_normal((len(proj_l), nr))
    tab[:, -1] = 0.0
    for n in (1, 31, 32, 33, 1000):
        g = rng.standard_normal((n, 3))
        pts = g / np.linalg.norm(g, axis=1)[:, None] * rng.uniform(0.0, 3.2, n)[:, None]   # some beyond the table (2.8)
        want = oracle_mod.projectors(pts, proj_l, tab, dr)
        for layout, mis in (("soa", 0), ("aos", 0), ("aos", 1), ("soa", 1)):
            got = gpu_projectors(sh, pts, proj_l, tab, dr, layout, misalign=mis)
            assert np.abs(got - want).max() <= TOL * max(1.0, np.abs(tab).max()), (n, layout, mis)
        for nvec in (1, 2, 5):   # segment kernel; ring kernel with four- and eight-vector consumers
            w = rng.standard_normal((nvec, n))
            coeff, abs_sum = oracle_mod.project(pts, proj_l, tab, dr, w)
            check_project(gpu_project(sh, pts, proj_l, tab, dr, w), coeff, abs_sum)


@pytest.mark.parametrize("proj_l", [[0], [1], [0, 1, 1], [2, 1], [4], [3, 3, 0], [7], [9, 9, 9, 9, 9, 4]])
def test_project_five_to_eight_vectors_column_tile_edges(sh, oracle_mod, proj_l):
    """5 to 8 weight vectors contract on the FP64 tensor-core instruction in tiles of 8 columns x 4 points: column counts of 1, 3, 7, 8, 9,
    15, 15 and 104 (one column, just below / at / just above a tile, the widest single pass), fewer vectors than the 8 rows of the instruction,
    one point, a ragged last 32-point tile, and enough tiles for every CTA of the persistent grid to wrap around its ring of slots."""
    rng = np.random.default_rng(900 + len(proj_l) * 17 + proj_l[0])
    nr, dr = 41, 0.08
    tab = rng.standard_normal((len(proj_l), nr))
    tab[:, -1] = 0.0
    for n in (1, 33, 4097, 148 * 32 * 9 + 5):
        g = rng.standard_normal((n, 3))
        pts = g / np.linalg.norm(g, axis=1)[:, None] * rng.uniform(0.0, 3.4, n)[:, None]
        for nvec in (5, 8):
            w = rng.standard_normal((nvec, n))
            coeff, abs_sum = oracle_mod.project(pts, proj_l, tab, dr, w)
            got = gpu_project(sh, pts, proj_l, tab, dr, w)
            check_project(got, coeff, abs_sum)
            assert np.array_equal(got, gpu_project(sh, pts, proj_l, tab, dr, w)), (n, nvec)   # fixed summation order


@pytest.mark.parametrize("proj_l", [[2], [0, 1, 3], [1, 1], [0, 2, 1, 3], [9, 9, 9, 4, 0], [0, 1, 2, 3, 4, 5, 6, 7, 8, 9], [5, 4, 4, 7], [9] * 11, [9] * 12])
def test_aos_store_modes(sh, oracle_mod, proj_l):
    """AoS copy-out modes of sh_projectors: odd ncols (one bulk copy per tile), even ncols with ncols/2 odd or even (one
    bulk copy per row, padded pitch), rows too wide for the bulk tile (12 x 19 = 228 columns), a misaligned `out` (warp copy);
    full tiles, a ragged tail and fewer points than one tile; one, two or four warps per tile (each evaluating part of the
    l-blocks)."""
    rng = np.random.default_rng(len(proj_l) * 31 + proj_l[0])
    nr, dr = 33, 0.1
    tab = rng.standard_normal((len(proj_l), nr))
    tab[:, -1] = 0.0
    for n in (7, 64, 1000 + 13):
        g = rng.standard_normal((n, 3))
        pts = g / np.linalg.norm(g, axis=1)[:, None] * rng.uniform(0.0, 3.5, n)[:, None]
        want = oracle_mod.projectors(pts, proj_l, tab, dr)
        for mis in (0, 1, 2):
            for mode in (0, 1, 2, 3):   # automatic, then each copy-out forced (where it applies)
                for split in (0, 1, 2, 4):   # warps sharing a tile (lmax >= 4): default, then each forced
                    ref = None
                    for pairs in ((0, 1) if split in (0, 1) else (0,)):   # 16-byte staging stores where the rows allow (default), or 8-byte always
                        sh.set_tuning("proj_aos_mode", mode)
                        sh.set_tuning("proj_aos_split", split)
                        sh.set_tuning("proj_aos_pairs", pairs)
                        try:
                            got = gpu_projectors(sh, pts, proj_l, tab, dr, "aos", misalign=mis)
                        finally:
                            sh.set_tuning("proj_aos_mode", 0)
                            sh.set_tuning("proj_aos_split", 0)
                            sh.set_tuning("proj_aos_pairs", 0)
                        assert np.abs(got - want).max() <= TOL * max(1.0, np.abs(tab).max()), (n, mis, mode, split, pairs)
                        if ref is None:
                            ref = got
                        assert np.array_equal(got, ref), (n, mis, mode, split, pairs)   # same arithmetic, different staging stores


@pytest.mark.parametrize("form", [1, 2])
def test_project_polynomial_forms_value_by_value(sh, oracle_mod, form):
    """sh_project has two polynomial forms (`project_form` knob): Horner in z^2 + the (x + iy)^m recurrence (1, the
    default of this FP64-bound call) and the factorized forms of every other call (2).  One-hot weight vectors turn the projection into the per-point values (every other term
    of the sum is an exact 0), so each form is checked VALUE BY VALUE against the oracle at the fp64 tolerance: random
    directions, points within 1e-6 of the poles and the axes, the origin, points beyond the table."""
    rng = np.random.default_rng(17)
    n = 96
    g = rng.standard_normal((n, 3))
    g[:24, :2] *= 1e-6          # near the poles
    g[24:36, 2] *= 1e-7         # near the equator (z ~ 0: the odd polynomials' zero)
    g[36:44, 1] *= 1e-9         # near the x axis
    pts = g / np.linalg.norm(g, axis=1)[:, None] * rng.uniform(0.05, 3.1, n)[:, None]
    pts[44] = 0.0
    pts[45] = (0.0, 0.0, -1.25)
    proj_l = [9, 0, 8, 1, 7, 2, 6, 3, 5, 4, 9]
    nr, dr = 31, 0.1
    tab = rng.standard_normal((len(proj_l), nr))
    tab[:, -1] = 0.0
    want = oracle_mod.projectors(pts, proj_l, tab, dr)          # [n][ncols]
    sh.set_tuning("project_form", form)
    try:
        got = gpu_project(sh, pts, proj_l, tab, dr, np.eye(n))   # coeff[v][col] = beta_col(point v)
    finally:
        sh.set_tuning("project_form", 0)
    err = np.abs(got - want).max()
    print(f"project_form {form}: max |beta_gpu - beta_oracle| = {err:.2e}")
    assert err <= TOL * max(1.0, np.abs(tab).max())


@pytest.mark.parametrize("nvec", [1, 4, 8])
def test_project_factorized_forms_full_grid(sh, oracle_mod, nvec):
    """The factorized forms (knob value 2; the default is Horner / recurrence) on the bench's FP64-bound workload (128^3 grid,
    100 columns) against the oracle's sum."""
    from paper_2510_05282_b200 import inputs

    pts = inputs.config3_full_grid()
    proj_l, tab, dr = inputs.projector_channels(lmax=9, per_l=1, cutoff=6.0, dr=0.02)
    w = inputs.wave_weights(len(pts), nvec, seed=8, volume_element=(12.0 / 128) ** 3)
    coeff, abs_sum = oracle_mod.project(pts, proj_l, tab, dr, w)
    sh.set_tuning("project_form", 2)
    try:
        got = gpu_project(sh, pts, proj_l, tab, dr, w)
    finally:
        sh.set_tuning("project_form", 0)
    check_project(got, coeff, abs_sum)


def test_many_channels_wide_rows(sh, oracle_mod):
    """32 channels of l = 9: 608 columns -- the AoS tile is 156 KB (one warp per CTA) and the projection runs as five
    launches of at most 128 columns."""
    rng = np.random.default_rng(7)
    proj_l = [9] * 32
    nr, dr = 41, 0.1
    tab = rng.standard_normal((32, nr))
    tab[:, -1] = 0.0
    n = 3000
    g = rng.standard_normal((n, 3))
    pts = g / np.linalg.norm(g, axis=1)[:, None] * rng.uniform(0.0, 4.0, n)[:, None]
    want = oracle_mod.projectors(pts, proj_l, tab, dr)
    for layout in ("soa", "aos"):
        assert np.abs(gpu_projectors(sh, pts, proj_l, tab, dr, layout) - want).max() <= TOL * np.abs(tab).max()
    w = rng.standard_normal((5, n))
    coeff, abs_sum = oracle_mod.project(pts, proj_l, tab, dr, w)
    check_project(gpu_project(sh, pts, proj_l, tab, dr, w), coeff, abs_sum)


def test_special_points_nodes_cutoff_origin_and_extremes(sh, oracle_mod):
    proj_l = [0, 1, 2, 0, 3]
    nr, dr = 33, 0.125                      # dr a power of two: nodes j*dr are exact
    rng = np.random.default_rng(9)
    tab = rng.standard_normal((len(proj_l), nr))
    rows = [[0.0, 0.0, 0.0], [-0.0, 0.0, -0.0]]
    for j in range(0, nr + 3):              # on nodes and midpoints, along axes and a diagonal, up to beyond the table
        for half in (0.0, 0.5):
            rr = (j + half) * dr
            if abs(rr - (nr - 1) * dr) < 1e-9:
                continue                    # the table's end is a discontinuity for a table that does not end with 0
            rows += [[rr, 0, 0], [0, -rr, 0], [0, 0, rr], [rr * 0.6, 0.0, rr * 0.8]]
    rows += [[1e-200, 2e-200, -1e-200], [1e-320, 0.0, 0.0], [3e200, 1e200, -2e200], [1.7e308, 1.7e308, 1.7e308]]
    pts = np.array(rows, dtype=np.float64)
    want = oracle_mod.projectors(pts, proj_l, tab, dr)
    for layout in ("soa", "aos"):
        got = gpu_projectors(sh, pts, proj_l, tab, dr, layout)
        assert np.abs(got - want).max() <= TOL * np.abs(tab).max()
    # r = 0: only the l = 0 channels survive, with the table's first entry
    got = gpu_projectors(sh, pts[:2], proj_l, tab, dr, "aos")
    y00 = 1.0 / np.sqrt(4.0 * np.pi)
    for row in got:
        assert abs(row[0] - tab[0, 0] * y00) <= 1e-15 and abs(row[9] - tab[3, 0] * y00) <= 1e-15
        assert np.all(np.delete(row, [0, 9]) == 0.0)
    # beyond the table: exact zeros
    far = np.array([[4.0, 0.1, 0.2], [1e10, 0.0, 0.0], [3e200, 1e200, -2e200]])
    assert np.all(gpu_projectors(sh, far, proj_l, tab, dr, "soa") == 0.0)
    # NaN coordinates (not an error): every l >= 1 column of that point is NaN, as in sh_real; the l = 0 columns are 0
    # (|r| is not inside the table); the other rows are untouched
    bad = pts[:6].copy()
    bad[2, 1] = np.nan
    got = gpu_projectors(sh, bad, proj_l, tab, dr, "soa")
    assert np.isnan(np.delete(got[2], [0, 9])).all() and np.all(got[2, [0, 9]] == 0.0)
    assert not np.isnan(np.delete(got, 2, axis=0)).any()


def test_empty_inputs(sh):
    import torch

    t = torch.ones((2, 4), dtype=torch.float64, device="cuda")
    x0 = torch.empty((0, 3), dtype=torch.float64, device="cuda")
    assert sh.sh_projectors(x0, [0, 1], t, 0.1, layout="aos").shape == (0, 4)
    c = sh.sh_project(x0, [0, 1], t, 0.1, torch.empty((2, 0), dtype=torch.float64, device="cuda"))
    torch.cuda.synchronize()
    assert c.shape == (2, 4) and torch.all(c == 0)
    # no channels: nothing to write
    x = torch.zeros((5, 3), dtype=torch.float64, device="cuda")
    assert sh.sh_projectors(x, [], torch.empty((0, 4), dtype=torch.float64, device="cuda"), 0.1).numel() == 0
    # workspace too small is refused
    with pytest.raises(sh.ShError):
        sh.sh_project(x, [0, 1], t, 0.1, torch.ones((1, 5), dtype=torch.float64, device="cuda"),
                      workspace=torch.empty(8, dtype=torch.uint8, device="cuda"))


def test_full_grid_moments_lmax9(sh, oracle_mod):
    """The bench's FP64-bound workload: the 128^3 grid (2,097,152 points), one channel per l <= 9 (100 columns), cutoff 6.0
    (grid corners reach r = 10.4: beyond the table).  The projection is compared for every column against the oracle's
    plain long-double sum over ALL points; the stored variant on every 41st point."""
    from paper_2510_05282_b200 import inputs

    pts = inputs.config3_full_grid()
    proj_l, tab, dr = inputs.projector_channels(lmax=9, per_l=1, cutoff=6.0, dr=0.02)
    w = inputs.wave_weights(len(pts), 8, seed=8, volume_element=(12.0 / 128) ** 3)
    coeff, abs_sum = oracle_mod.project(pts, proj_l, tab, dr, w)
    # one vector: segment kernel; two and four: ring kernel with DFMA consumers; eight: ring kernel contracting on the FP64 tensor-core instruction
    for nvec in (1, 2, 4, 8):
        got = gpu_project(sh, pts, proj_l, tab, dr, w[:nvec])
        worst = check_project(got, coeff[:nvec], abs_sum[:nvec])
        print(f"full grid projection, {nvec} vectors: max |c_gpu - c_oracle| / sum|terms| = {worst:.2e}")
    import torch

    x = torch.from_numpy(pts).cuda()
    t = torch.from_numpy(tab).cuda()
    sel = np.arange(0, len(pts), 41)
    want = oracle_mod.projectors(pts[sel], proj_l, tab, dr)
    for layout in ("soa", "aos"):
        out = sh.sh_projectors(x, proj_l, t, dr, layout=layout)
        torch.cuda.synchronize()
        res = out[:, torch.from_numpy(sel).cuda()].T if layout == "soa" else out[torch.from_numpy(sel).cuda()]
        assert np.abs(res.cpu().numpy() - want).max() <= TOL * max(1.0, np.abs(tab).max())
        del out
