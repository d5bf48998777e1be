"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (symmetric kernels, two voxels
per thread in the back-projector, three multi-grid levels), through the C ABI.

* config 3 (256^3, 40 views of 512x384): P and P^T element by element against the whole oracle, the adjoint
  identity, a multi-step TV-prox call, and a 3-level reconstruction with reduced iteration counts.
* config 2 (128^3, 40 views of 256x192, noisy data): 2-level reconstruction with reduced iteration counts.
* config 4 (512x512x256, 360 views): too large for the whole oracle in minutes -> SAMPLED outputs the oracle
  computes one by one: P on sampled views (an oracle geometry holding only those angles), P^T on sampled
  16^3 blocks of voxels (an oracle geometry whose volume IS that block, offset to the same voxel centres:
  a(ray, voxel) depends on the voxel's position only, so its back-projection equals the full one there).
"""
import numpy as np
import pytest

from paper_1001_0599_b200 import inputs as I

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

TOL_PROJ = 1e-5
TOL_VOL = 1e-3


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (run with -m 'not gpu' on CPU boxes)")
    return torch


@pytest.fixture(scope="module")
def cbct(torch):
    from paper_1001_0599_b200 import cbct
    cbct.load_library()
    return cbct


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def block_geometry(g, i0, j0, k0, n=16):
    """The oracle geometry whose whole volume is voxels [i0,i0+n) x [j0,j0+n) x [k0,k0+n) of g."""
    off = (g.vol_off[0] + (i0 + 0.5 * (n - 1) - 0.5 * (g.nx - 1)) * g.hx,
           g.vol_off[1] + (j0 + 0.5 * (n - 1) - 0.5 * (g.ny - 1)) * g.hy,
           g.vol_off[2] + (k0 + 0.5 * (n - 1) - 0.5 * (g.nz - 1)) * g.hz)
    return g.replace(nx=n, ny=n, nz=n, vol_off=off, angles=g.angles_rad())


def test_config3_projectors_full_size(torch, cbct, orc):
    g = I.config(3).geom
    f = I.uniform_volume(g, 31)
    q = I.uniform_projections(g, 32)
    with cbct.geometry_create(g, max_levels=3) as h:
        assert h.symmetry == 8
        p = torch.empty(g.proj_shape, device="cuda", dtype=torch.float32)
        b = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
        h.forward_project(dev(torch, f), p)
        h.back_project(dev(torch, q), b)
        got_p, got_b = p.cpu().numpy(), b.cpu().numpy()
        h.forward_project(dev(torch, f), p)
        h.back_project(dev(torch, q), b)
        assert p.cpu().numpy().tobytes() == got_p.tobytes() and b.cpu().numpy().tobytes() == got_b.tobytes()
    want_p = orc.forward(g, f)
    for a in range(g.n_proj):
        assert rel_l2(got_p[a], want_p[a]) <= TOL_PROJ, (a, rel_l2(got_p[a], want_p[a]))
    want_b = orc.back(g, q)
    assert rel_l2(got_b, want_b) <= TOL_PROJ, rel_l2(got_b, want_b)
    assert np.abs(got_b - want_b).max() <= 1e-4 * np.abs(want_b).max()
    lhs = np.vdot(got_p.astype(np.float64), (q - 0.3).astype(np.float64))
    rhs = np.vdot(f.astype(np.float64), got_b.astype(np.float64)) - 0.3 * got_p.astype(np.float64).sum()
    # <P f, q - 0.3> = <f, P^T q> - 0.3 <P f, 1>: the adjoint identity with a sign-changing test vector
    assert abs(lhs - rhs) <= 1e-5 * abs(np.vdot(got_p.astype(np.float64), q.astype(np.float64)))


def test_config3_tv_prox_full_size(torch, cbct, orc):
    cfg = I.config(3)
    g = cfg.geom
    gg = (I.paint(cfg.ellipsoids, g) + 0.002 * (I.uniform_volume(g, 33, hi=1.0) - 0.5)).astype(np.float32)
    setup = I.FbsSetup(max_inner=4, rel_tol=0.0)
    w = 2.0e-5
    want, wrep = orc.tv_prox(g, gg, w, setup)
    with cbct.geometry_create(g) as h:
        f = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
        rep = h.tv_prox(dev(torch, gg), f, w, setup)
        got = f.cpu().numpy()
    assert (rep.inner_iters, rep.trials) == (wrep.inner_iters, wrep.trials)
    assert rel_l2(got, want) <= 1e-5
    assert rel_l2(got - gg, want - gg) <= 1e-3
    assert rep.e_last == pytest.approx(wrep.e_last, rel=1e-6)


@pytest.mark.parametrize("k,iters", [(2, (3, 2))])
def test_fbs_reduced_counts_at_full_size(torch, cbct, orc, k, iters):
    """Config 2 as stated (sizes, noise, levels) with reduced iteration counts per level, run twice (bitwise)."""
    cfg = I.config(k)
    g = cfg.geom
    y = I.make_projections(cfg)
    setup = I.FbsSetup(**{**cfg.fbs.__dict__, "iters_per_level": iters})
    want = orc.fbs(g, y, setup)
    with cbct.geometry_create(g, max_levels=len(iters)) as h:
        f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        rep = h.fbs_reconstruct(dev(torch, y), f, setup)
        got = f.cpu().numpy()
        f.zero_()
        h.fbs_reconstruct(dev(torch, y), f, setup)
        assert f.cpu().numpy().tobytes() == got.tobytes()
    assert rel_l2(got, want.f) <= TOL_VOL, rel_l2(got, want.f)
    np.testing.assert_allclose(rep.objective, want.objective, rtol=1e-4)
    np.testing.assert_allclose(rep.step_abs, want.step_abs, rtol=1e-5)


def test_config4_sampled_outputs(torch, cbct, orc):
    g = I.config(4).geom
    f = I.uniform_volume(g, 41)
    q = I.uniform_projections(g, 42)
    with cbct.geometry_create(g) as h:
        assert h.symmetry == 8
        p = torch.empty(g.proj_shape, device="cuda", dtype=torch.float32)
        h.forward_project(dev(torch, f), p)
        views = [0, 37, 90, 151, 233, 359]
        got_p = p[views].cpu().numpy()
        del p
        b = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
        h.back_project(dev(torch, q), b)
        got_b = b.cpu().numpy()
    gs = g.replace(n_proj=len(views), angles=g.angles_rad()[views])
    want_p = orc.forward(gs, f)
    for n, a in enumerate(views):
        assert rel_l2(got_p[n], want_p[n]) <= TOL_PROJ, (a, rel_l2(got_p[n], want_p[n]))
    scale = np.abs(got_b).max()
    for (i0, j0, k0) in [(0, 0, 0), (248, 248, 120), (496, 0, 240), (131, 377, 5), (300, 200, 128)]:
        want = orc.back(block_geometry(g, i0, j0, k0), q)
        blk = got_b[k0:k0 + 16, j0:j0 + 16, i0:i0 + 16]
        assert rel_l2(blk, want) <= TOL_PROJ, ((i0, j0, k0), rel_l2(blk, want))
        assert np.abs(blk - want).max() <= 1e-4 * scale


def test_config2_as_stated_full_iteration_counts(torch, cbct, orc):
    """Config 2 of BASELINE.json exactly as stated: 128^3, 40 noisy views of 256x192, 50 FBS iterations on each of
    2 multi-grid levels, against the whole oracle reconstruction (about a minute of host time)."""
    cfg = I.config(2)
    g = cfg.geom
    y = I.make_projections(cfg)
    want = orc.fbs(g, y, cfg.fbs)
    with cbct.geometry_create(g, max_levels=2) as h:
        f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        rep = h.fbs_reconstruct(dev(torch, y), f, cfg.fbs)
        got = f.cpu().numpy()
    assert rep.n_iters_total == 100
    assert rel_l2(got, want.f) <= TOL_VOL, rel_l2(got, want.f)
    np.testing.assert_allclose(rep.objective, want.objective, rtol=1e-4)
    assert np.all(rep.objective[1:50] <= rep.objective[:49] * (1 + 1e-6))      # monotone within a level
    assert np.all(rep.objective[51:] <= rep.objective[50:-1] * (1 + 1e-6))
    # S18: every Armijo / stop decision of the 100 prox calls falls the same way in fp32 sums as in fp64
    assert (rep.inner_total, rep.trials_total) == (want.inner_total, want.trials_total)


def test_config3_as_stated_full_coarse_levels_ten_finest_iterations(torch, cbct, orc):
    """Config 3 of BASELINE.json as stated -- 256^3, 40 noisy views of 512x384, 3 multi-grid levels, 100 iterations on
    each of the two coarse levels -- and 10 of the 100 finest-level iterations (the whole oracle run of those 210
    iterations is a few minutes of host time; the remaining 90 finest iterations repeat the same kernels on the same
    sizes).  Volume <= 1e-3, objective series 1e-4, identical Armijo counts, bitwise repeatable."""
    cfg = I.config(3)
    g = cfg.geom
    y = I.make_projections(cfg)
    setup = I.FbsSetup(**{**cfg.fbs.__dict__, "iters_per_level": (100, 100, 10)})
    want = orc.fbs(g, y, setup)
    with cbct.geometry_create(g, max_levels=3) as h:
        assert [h.back_path(l) for l in range(3)] == ["tma", "tma", "tma"]
        f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        rep = h.fbs_reconstruct(dev(torch, y), f, setup)
        got = f.cpu().numpy()
        f.zero_()
        h.fbs_reconstruct(dev(torch, y), f, setup, objective=False)          # the look-ahead path of the bench
        assert f.cpu().numpy().tobytes() == got.tobytes()
        assert h.bound_violations() == 0
    assert rep.n_iters_total == 210
    assert rel_l2(got, want.f) <= TOL_VOL, rel_l2(got, want.f)
    np.testing.assert_allclose(rep.objective, want.objective, rtol=1e-4)
    np.testing.assert_allclose(rep.step_abs, want.step_abs, rtol=1e-5)
    assert (rep.inner_total, rep.trials_total) == (want.inner_total, want.trials_total)


def test_config4_tv_prox_step_bound_and_one_iteration_per_level(torch, cbct, orc):
    """Config 4 as stated (512x512x256 at 0.5 x 0.5 x 1 mm, 360 noisy views, 3 levels) through everything but the
    iteration count: one TV-prox call of 4 descent steps on the whole anisotropic volume, and a (1, 1, 1) reconstruction
    compared on the WHOLE volume -- its report carries tau = step / Lhat of every level, i.e. cbct_step_bound at full
    size.  One finest-level oracle iteration (P, P^T on 360 views, twice: Lhat and the iteration) is minutes of host time."""
    cfg = I.config(4)
    g = cfg.geom
    gg = (I.paint(cfg.ellipsoids, g) + 0.002 * (I.uniform_volume(g, 43, hi=1.0) - 0.5)).astype(np.float32)
    tvs = I.FbsSetup(max_inner=4, rel_tol=0.0)
    w = 2.0e-5
    want_tv, wrep = orc.tv_prox(g, gg, w, tvs)
    y = I.make_projections(cfg)
    setup = I.FbsSetup(**{**cfg.fbs.__dict__, "iters_per_level": (1, 1, 1)})
    want = orc.fbs(g, y, setup)
    with cbct.geometry_create(g, max_levels=3) as h:
        f = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
        rep = h.tv_prox(dev(torch, gg), f, w, tvs)
        got_tv = f.cpu().numpy()
        f.zero_()
        frep = h.fbs_reconstruct(dev(torch, y), f, setup)
        got = f.cpu().numpy()
        lhat = h.step_bound()
        assert h.bound_violations() == 0
    assert (rep.inner_iters, rep.trials) == (wrep.inner_iters, wrep.trials)
    assert rel_l2(got_tv, want_tv) <= 1e-5
    assert rel_l2(got_tv - gg, want_tv - gg) <= 1e-3
    assert rep.e_last == pytest.approx(wrep.e_last, rel=1e-6)
    assert rel_l2(got, want.f) <= TOL_VOL, rel_l2(got, want.f)
    np.testing.assert_allclose(frep.objective, want.objective, rtol=1e-4)
    np.testing.assert_allclose(frep.step_abs, want.step_abs, rtol=1e-5)
    assert cfg.fbs.step / lhat == pytest.approx(want.step_abs[-1], rel=1e-5)
    assert (frep.inner_total, frep.trials_total) == (want.inner_total, want.trials_total)


def test_config4_back_projector_blocks_at_the_detector_edge(torch, cbct, orc):
    """Two more sampled 16^3 blocks of config 4, where the cone clips the volume in v (top and bottom slices)."""
    g = I.config(4).geom
    q = I.uniform_projections(g, 42)
    with cbct.geometry_create(g) as h:
        b = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
        h.back_project(dev(torch, q), b)
        got_b = b.cpu().numpy()
    scale = np.abs(got_b).max()
    for (i0, j0, k0) in [(248, 248, 20), (60, 420, 232)]:
        want = orc.back(block_geometry(g, i0, j0, k0), q)
        blk = got_b[k0:k0 + 16, j0:j0 + 16, i0:i0 + 16]
        assert np.abs(want).max() > 0 and (want == 0).any()          # the block straddles the edge of the cone
        assert rel_l2(blk, want) <= TOL_PROJ, ((i0, j0, k0), rel_l2(blk, want))
        assert np.abs(blk - want).max() <= 1e-4 * scale
        assert np.array_equal(blk == 0.0, want == 0.0)


# ---------------------------------------------------------------------------
# config 5: the operator sweep's extreme cases against the oracle (inputs of inputs.uniform_*: bench.py --sweep uses the same)
# ---------------------------------------------------------------------------

def test_config5_smallest_case_whole_operators(torch, cbct, orc):
    """64^3 at 4 mm, ONE view of 512x384: a voxel's shadow is ~8 pixels wide (the general gather kernel)."""
    g = I.sweep_geometry(64, 1)
    f = I.uniform_volume(g, I.SEED_BASE + 5, hi=0.03)
    q = I.uniform_projections(g, I.SEED_BASE + 6)
    with cbct.geometry_create(g) as h:
        assert h.back_path(0) == "gather"
        p = torch.empty(g.proj_shape, device="cuda", dtype=torch.float32)
        b = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
        h.forward_project(dev(torch, f), p)
        h.back_project(dev(torch, q), b)
        got_p, got_b = p.cpu().numpy(), b.cpu().numpy()
        S = h.count_samples()
    want_p, S_want = orc.forward(g, f, return_samples=True)
    want_b = orc.back(g, q)
    assert rel_l2(got_p[0], want_p[0]) <= TOL_PROJ
    assert rel_l2(got_b, want_b) <= TOL_PROJ
    assert np.abs(got_b - want_b).max() <= 1e-4 * np.abs(want_b).max()
    assert abs(S - S_want) <= 2e-3 * S_want


def test_config5_largest_case_sampled_outputs(torch, cbct, orc):
    """512^3 at 0.5 mm, 360 views of 512x384: a voxel's shadow is ~1 pixel.  P on 3 sampled views, P^T on 3 sampled
    16^3 blocks (an oracle geometry whose volume IS the block)."""
    g = I.sweep_geometry(512, 360)
    f = I.uniform_volume(g, I.SEED_BASE + 5, hi=0.03)
    q = I.uniform_projections(g, I.SEED_BASE + 6)
    with cbct.geometry_create(g) as h:
        assert h.symmetry == 8
        p = torch.empty(g.proj_shape, device="cuda", dtype=torch.float32)
        h.forward_project(dev(torch, f), p)
        views = [3, 134, 271]
        got_p = p[views].cpu().numpy()
        del p
        b = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
        h.back_project(dev(torch, q), b)
        got_b = b.cpu().numpy()
        del b
    gs = g.replace(n_proj=len(views), angles=g.angles_rad()[views])
    want_p = orc.forward(gs, f)
    for n, a in enumerate(views):
        assert rel_l2(got_p[n], want_p[n]) <= TOL_PROJ, (a, rel_l2(got_p[n], want_p[n]))
    scale = np.abs(got_b).max()
    for (i0, j0, k0) in [(7, 490, 250), (255, 249, 60), (400, 130, 470)]:
        want = orc.back(block_geometry(g, i0, j0, k0), q)
        blk = got_b[k0:k0 + 16, j0:j0 + 16, i0:i0 + 16]
        assert rel_l2(blk, want) <= TOL_PROJ, ((i0, j0, k0), rel_l2(blk, want))
        assert np.abs(blk - want).max() <= 1e-4 * scale
