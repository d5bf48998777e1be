"""Pins of the oracle's FBS iteration and multi-grid driver."""
import numpy as np
import pytest

from paper_1001_0599_b200 import inputs as I


def tiny(n=16, n_proj=6, nu=24):
    return I.Geometry(nx=n, ny=n, nz=n, hx=64.0 / n, hy=64.0 / n, hz=64.0 / n, nu=nu, nv=nu,
                      du=76.8 / nu, dv=76.8 / nu, sad=1000.0, sdd=1500.0, n_proj=n_proj)


def test_P14_tv_off_is_landweber(orc):
    """tv_weight = 0, clip off: f <- f - tau c_norm P^T(P f - y), written out here from P, P^T."""
    g = tiny()
    rng = np.random.default_rng(0)
    y = orc.forward(g, rng.random(g.vol_shape) * 0.02)
    setup = I.FbsSetup(tv_weight=0.0, step=0.9, iters_per_level=(4,), nonneg=False)
    res = orc.fbs(g, y, setup)
    c_norm = 2.0 * g.nx * g.ny * g.nz / (g.n_proj * g.nu * g.nv)
    q = orc.back(g, orc.forward(g, np.ones(g.vol_shape)))
    tau = 0.9 / (c_norm * q.max())
    f = np.zeros(g.vol_shape)
    obj = []
    for _ in range(4):
        T = orc.forward(g, f) - y
        obj.append((T ** 2).mean())
        f = f - tau * c_norm * orc.back(g, T)
    np.testing.assert_allclose(res.f, f, rtol=0, atol=1e-15)
    np.testing.assert_allclose(res.objective, obj, rtol=1e-13)
    assert res.step_abs[0] == pytest.approx(tau, rel=1e-14)
    assert res.objective[-1] < res.objective[0]


def test_P12_row_sum_bound_dominates_power_iteration(orc):
    g = tiny(n=12, n_proj=5, nu=20)
    c_norm = 2.0 * g.nx * g.ny * g.nz / (g.n_proj * g.nu * g.nv)
    Lhat = orc.step_bound(g)
    x = np.random.default_rng(1).random(g.vol_shape)
    lam = 0.0
    for _ in range(50):
        x /= np.linalg.norm(x)
        z = c_norm * orc.back(g, orc.forward(g, x))
        lam = np.vdot(x, z)
        x = z
    assert lam <= Lhat * (1 + 1e-12)
    assert lam > 0.2 * Lhat          # the bound is not vacuous


def test_P11_objective_is_non_increasing_on_config1_shape(orc):
    """Config-1-like case, noiseless analytic data (L145-L151; convexity L215): with step <= 1
    J = tv_weight E1 + E2 does not increase, and E2 falls by a large factor."""
    g = tiny(n=16, n_proj=8, nu=24)
    ell = I.headlike_phantom(32.0)
    y = I.analytic_projections(ell, g)
    setup = I.FbsSetup(tv_weight=0.01, step=1.0, iters_per_level=(12,))
    res = orc.fbs(g, y, setup)
    J = res.objective
    assert np.all(J[1:] <= J[:-1] * (1 + 1e-6)), J
    assert J[-1] < 0.05 * J[0]
    assert res.f.min() >= 0.0
    truth = I.paint(ell, g)
    err0 = np.linalg.norm(truth)
    assert np.linalg.norm(res.f - truth) < 0.8 * err0


def test_multigrid_driver_structure(orc):
    """Two levels == (bin data, solve coarse from zeros, prolong, solve fine from that),
    assembled here from the oracle's single-level pieces; S12/S13 are design choices
    (parity unpinned) -- this pins only the wiring and the level geometry."""
    g = tiny(n=16, n_proj=6, nu=24)
    ell = I.headlike_phantom(32.0)
    y = I.analytic_projections(ell, g)
    two = orc.fbs(g, y, I.FbsSetup(iters_per_level=(5, 3)))
    gc = g.replace(nx=8, ny=8, nz=8, hx=8.0, hy=8.0, hz=8.0, nu=12, nv=12, du=6.4, dv=6.4)
    coarse = orc.fbs(gc, orc.bin2(y), I.FbsSetup(iters_per_level=(5,)))
    start = orc.prolong(coarse.f, g.bc_xy, g.bc_z)
    fine = orc.fbs(g, y, I.FbsSetup(iters_per_level=(3,)), f0=start)
    np.testing.assert_allclose(two.f, fine.f, rtol=0, atol=1e-15)
    np.testing.assert_allclose(two.objective, np.concatenate([coarse.objective, fine.objective]), rtol=1e-13)
    # the coarse level's pixel centres are the means of the fine pairs: a binned ANALYTIC
    # projection is close to the analytic projection of the coarse geometry
    ya = I.analytic_projections(ell, gc)
    err = np.linalg.norm(orc.bin2(y) - ya)
    assert err < 0.12 * np.linalg.norm(ya)
    for du_, dv_ in ((3.2, 0.0), (0.0, 3.2), (-3.2, 0.0)):       # half a coarse pixel off: worse
        yb = I.analytic_projections(ell, gc.replace(det_off_u=du_, det_off_v=dv_))
        assert np.linalg.norm(orc.bin2(y) - yb) > 1.5 * err
    # a supplied initial volume is restricted to the coarsest level first
    f0 = I.paint(ell, g).astype(np.float64)
    a = orc.fbs(g, y, I.FbsSetup(iters_per_level=(2, 1)), f0=f0)
    cb = orc.fbs(gc, orc.bin2(y), I.FbsSetup(iters_per_level=(2,)), f0=orc.restrict(f0))
    b = orc.fbs(g, y, I.FbsSetup(iters_per_level=(1,)), f0=orc.prolong(cb.f, g.bc_xy, g.bc_z))
    np.testing.assert_allclose(a.f, b.f, rtol=0, atol=1e-15)


def test_convergence_stopping_is_the_fixed_count_run_cut_at_the_first_small_change(orc):
    """NEXT-2, 'until convergence' (reading S20): with conv_tol the level stops after the first
    iteration whose relative change ||f_new - f_old|| / ||f_old|| is <= conv_tol.  Pinned against runs with FIXED
    counts (which do not execute the test): the stopped run equals the n-iteration run, its last change is below the
    tolerance and every earlier change above it."""
    cfg = I.config(1)
    y = I.make_projections(cfg)
    tol = 0.05
    r = orc.fbs(cfg.geom, y, I.FbsSetup(iters_per_level=(40,), conv_tol=tol))
    n = r.iters_done[0]
    assert 2 < n < 40 and len(r.objective) == n
    runs = [orc.fbs(cfg.geom, y, I.FbsSetup(iters_per_level=(m,))).f for m in range(1, n + 1)]
    assert np.array_equal(r.f, runs[-1])
    change = [np.linalg.norm(runs[m] - runs[m - 1]) / np.linalg.norm(runs[m - 1]) for m in range(1, n)]
    assert change[-1] <= tol and all(c > tol for c in change[:-1])
