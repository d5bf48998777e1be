"""Pins of the oracle's geometry and projectors -- CPU only.

Nothing here compares the oracle with itself through the same routine: each test
holds it to a closed form, a hand value, an invariant or brute force."""
import os

import numpy as np
import pytest

from paper_1001_0599_b200 import inputs as I

HERE = os.path.dirname(os.path.abspath(__file__))


def small_geom(n=(10, 12, 8), h=(2.0, 1.5, 2.5), nu=14, nv=10, du=3.1, n_proj=5, angles=None,
               off=(0.7, -1.1, 0.4), det_off=(0.3, -0.2)):
    return I.Geometry(nx=n[0], ny=n[1], nz=n[2], hx=h[0], hy=h[1], hz=h[2], nu=nu, nv=nv, du=du,
                      dv=du * 1.1, sad=200.0, sdd=320.0, n_proj=n_proj, vol_off=off,
                      det_off_u=det_off[0], det_off_v=det_off[1], angles=angles)


def test_hand_ray_box_lengths(orc):
    """tests/golden/ray_box_hand.txt: lengths derived by hand."""
    rows = 0
    for line in open(os.path.join(HERE, "golden", "ray_box_hand.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        v = [float(x) for x in line.split()]
        got = orc.ray_box_len(v[0:3], v[3:6], v[6:9], v[9:12])
        assert got == pytest.approx(v[12], abs=1e-13), line
        rows += 1
    assert rows == 9


def test_geometry_theta0_is_appendix_A2_A6(orc):
    """At theta=0: D = (L0, -u, v) = L n of Eq. A2 and the voxel->detector
    map is Eq. A6 (L401-L406) literally; l* = L(u*,v*) (x - x_S)/L0."""
    g = small_geom(angles=np.array([0.0]), n_proj=1)
    for iu, iv in [(0, 0), (3, 7), (13, 9)]:
        S, D = orc.ray(g, 0, iu, iv)
        u = (iu - (g.nu - 1) / 2) * g.du + g.det_off_u
        v = (iv - (g.nv - 1) / 2) * g.dv + g.det_off_v
        np.testing.assert_allclose(S, [-g.sad, 0, 0], atol=1e-13)
        np.testing.assert_allclose(D, [g.sdd, -u, v], atol=1e-13)
    X = np.array([12.5, -7.0, 9.0])
    us, vs, l = orc.voxel_to_detector(g, 0, X)
    xs, ys, zs = -g.sad, 0.0, 0.0
    assert us == pytest.approx(-(X[1] - ys) * g.sdd / (X[0] - xs), rel=1e-14)
    assert vs == pytest.approx((X[2] - zs) * g.sdd / (X[0] - xs), rel=1e-14)
    Lstar = np.sqrt(g.sdd ** 2 + us ** 2 + vs ** 2)
    assert l == pytest.approx(Lstar * (X[0] - xs) / g.sdd, rel=1e-14)


def test_ray_hits_the_voxel_it_was_mapped_from(orc):
    """(u*,v*) of A6 for a general angle: the ray to that detector point passes through X."""
    g = small_geom(n_proj=7)
    X = np.array([9.0, -4.0, 6.5])
    for a in range(g.n_proj):
        us, vs, l = orc.voxel_to_detector(g, a, X)
        th = g.angles_rad()[a]
        c, s = np.cos(th), np.sin(th)
        S = np.array([-g.sad * c, -g.sad * s, 0.0])
        P = S + g.sdd * np.array([c, s, 0]) + us * np.array([s, -c, 0]) + vs * np.array([0, 0, 1.0])
        t = l / np.linalg.norm(P - S)
        np.testing.assert_allclose(S + t * (P - S), X, atol=1e-10)


@pytest.mark.parametrize("angles", [
    np.deg2rad([0.0, 45.0, 90.0, 180.0, 270.0]),
    np.deg2rad([13.0, 101.5, 222.2, 359.0]),
])
def test_P1_traversal_equals_brute_force(orc, angles):
    g = small_geom(angles=angles, n_proj=len(angles))
    rng = np.random.default_rng(1)
    f = rng.random(g.vol_shape)
    pb = orc.forward_brute(g, f)
    pt, S = orc.forward(g, f, return_samples=True)
    assert np.abs(pb - pt).max() <= 1e-12 * max(1.0, np.abs(pb).max())
    assert pb.max() > 1.0
    # S counts the pairs with positive length: compare with a brute-force count on ones
    pbl = orc.forward_brute(g, np.ones(g.vol_shape))
    assert S > 0 and np.count_nonzero(pbl) <= g.n_proj * g.nu * g.nv


def test_P1_centred_even_grid_with_axis_aligned_views(orc):
    """Centred even grids put planes through the isocentre: the awkward case for ties."""
    g = I.Geometry(nx=8, ny=8, nz=8, hx=2.0, hy=2.0, hz=2.0, nu=12, nv=12, du=2.0, dv=2.0,
                   sad=100.0, sdd=150.0, n_proj=8)
    rng = np.random.default_rng(2)
    f = rng.random(g.vol_shape)
    np.testing.assert_allclose(orc.forward(g, f), orc.forward_brute(g, f), rtol=0, atol=1e-12)


def _chord_numpy(S, D, lo, hi):
    """Independent closed form of the chord of a segment in a box (numpy slab test)."""
    with np.errstate(divide="ignore", invalid="ignore"):
        t1 = (lo - S) / D
        t2 = (hi - S) / D
    tn = np.minimum(t1, t2).max()
    tf = np.maximum(t1, t2).min()
    return max(0.0, min(tf, 1.0) - max(tn, 0.0)) * np.linalg.norm(D)


def test_P2_constant_volume_gives_chord_of_bounding_box(orc):
    g = small_geom(n_proj=6)
    c = 0.37
    p = orc.forward(g, np.full(g.vol_shape, c))
    half = np.array([g.nx * g.hx, g.ny * g.hy, g.nz * g.hz]) / 2
    lo, hi = np.array(g.vol_off) - half, np.array(g.vol_off) + half
    for a in range(g.n_proj):
        for iv in range(g.nv):
            for iu in range(g.nu):
                S, D = orc.ray(g, a, iu, iv)
                assert p[a, iv, iu] == pytest.approx(c * _chord_numpy(S, D, lo, hi), abs=1e-11)
    assert p.max() > 0


def test_P3_voxelised_phantom_converges_to_analytic_integrals(orc):
    """Closed-form ellipsoid line integrals (unit-sphere transform): the Siddon projection of
    the centre-sampled phantom converges to them at first order in h (north_star pin).
    Piecewise-constant voxels are first-order accurate, so the error must roughly halve per
    refinement; a mirrored / transposed geometry would leave an O(1) error instead."""
    ell = I.headlike_phantom(32.0) + [I.Ellipsoid((9.0, -6.0, 4.0), (9.0, 14.0, 7.0), 0.4, 0.01)]
    errs = []
    for n in (16, 32, 64, 128):
        g = I.Geometry(nx=n, ny=n, nz=n, hx=64.0 / n, hy=64.0 / n, hz=64.0 / n, nu=24, nv=24,
                       du=3.2, dv=3.2, sad=1000.0, sdd=1500.0, n_proj=4)
        ana = I.analytic_projections(ell, g)
        num = orc.forward(g, I.paint(ell, g))
        errs.append(np.linalg.norm(num - ana) / np.linalg.norm(ana))
    assert errs[3] < 0.035, errs
    assert errs[2] < 0.7 * errs[1] and errs[3] < 0.7 * errs[2], errs
    # the mirrored phantom does NOT converge: the pin is sensitive to orientation
    g = I.Geometry(nx=64, ny=64, nz=64, hx=1.0, hy=1.0, hz=1.0, nu=24, nv=24, du=3.2, dv=3.2,
                   sad=1000.0, sdd=1500.0, n_proj=4)
    ana = I.analytic_projections(ell, g)
    for flipped in (I.paint(ell, g)[:, :, ::-1], np.transpose(I.paint(ell, g), (0, 2, 1))):
        bad = orc.forward(g, np.ascontiguousarray(flipped))
        assert np.linalg.norm(bad - ana) / np.linalg.norm(ana) > 3 * errs[2]


def test_P4_eq6_continuum_limit_of_the_transpose(orc):
    """Eq. 6 (Jacobian A7, L412): with a fine detector and smooth T,
    (du dv / dV) (P^T T)_v -> L^3(u*,v*) / (L0 l^2) T(u*,v*).
    The sum over rays is a Riemann sum of a function with sharp edges in v (voxel faces are
    parallel to e_v), so its error is O(dv / footprint): a 4 mm detector window of 800^2
    pixels centred on the voxel's (u*,v*) brings it to a few 1e-3."""
    h = 1.0
    base = dict(nx=6, ny=6, nz=6, hx=h, hy=h, hz=h, nu=800, nv=800, du=0.005, dv=0.005,
                sad=200.0, sdd=300.0, n_proj=1)
    Tfun = lambda uu, vv: 1.0 + 0.05 * uu - 0.03 * vv + 0.01 * uu * vv
    worst = 0.0
    for th, (i, j, k) in [(0.0, (2, 3, 1)), (37.0, (0, 5, 4)), (200.0, (3, 2, 3)), (90.0, (5, 0, 0))]:
        g = I.Geometry(angles=np.deg2rad([th]), **base)
        X = np.array([(i - 2.5) * h, (j - 2.5) * h, (k - 2.5) * h])
        us, vs, l = orc.voxel_to_detector(g, 0, X)
        g = g.replace(det_off_u=us, det_off_v=vs)
        u = (np.arange(g.nu) - (g.nu - 1) / 2) * g.du + us
        v = (np.arange(g.nv) - (g.nv - 1) / 2) * g.dv + vs
        U, V = np.meshgrid(u, v)
        b = orc.back(g, Tfun(U, V)[None])
        L = np.sqrt(g.sdd ** 2 + us ** 2 + vs ** 2)
        want = L ** 3 / (g.sdd * l ** 2) * Tfun(us, vs)
        got = g.du * g.dv / h ** 3 * b[k, j, i]
        worst = max(worst, abs(got / want - 1))
    assert worst < 0.01, worst


def test_P5_adjoint_identity(orc):
    g = small_geom(n_proj=6)
    rng = np.random.default_rng(3)
    f = rng.random(g.vol_shape)
    q = rng.random(g.proj_shape)
    lhs = np.vdot(orc.forward(g, f), q)
    rhs = np.vdot(f, orc.back(g, q))
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


def test_back_scatter_equals_brute_gather(orc):
    g = small_geom(n=(5, 6, 4), nu=9, nv=7, du=4.5, n_proj=3)
    rng = np.random.default_rng(4)
    q = rng.random(g.proj_shape)
    np.testing.assert_allclose(orc.back(g, q), orc.back_brute(g, q), rtol=0, atol=1e-11)


def test_P6_quarter_turn_symmetry(orc):
    """P_{theta+90deg}(f) = P_theta(f rotated by -90deg) on a centred cubic grid, hx = hy."""
    n = 10
    base = dict(nx=n, ny=n, nz=6, hx=2.0, hy=2.0, hz=3.0, nu=16, nv=8, du=2.5, dv=3.0,
                sad=150.0, sdd=260.0, n_proj=1)
    th = np.deg2rad(25.0)
    g0 = I.Geometry(angles=np.array([th]), **base)
    g1 = I.Geometry(angles=np.array([th + np.pi / 2]), **base)
    rng = np.random.default_rng(5)
    f = rng.random(g0.vol_shape)                # [z, y, x]
    # rotating the scanner by +90deg about z == rotating the object by -90deg:
    # f'(x, y) = f(-y, x)  ->  f'[k, j, i] = f[k, i, n-1-j]
    fr = np.transpose(f, (0, 2, 1))[:, :, ::-1].copy()
    fr2 = np.transpose(f, (0, 2, 1))[:, ::-1, :].copy()
    p1 = orc.forward(g1, f)
    cand = [orc.forward(g0, fr), orc.forward(g0, fr2)]
    errs = [np.abs(p1 - c).max() for c in cand]
    assert min(errs) < 1e-11 and max(errs) > 1e-3   # exactly one orientation matches


def test_truncated_detector_and_rays_missing_the_volume(orc):
    """Rays that miss give exactly 0; voxels seen by no ray back-project to exactly 0."""
    g = I.Geometry(nx=8, ny=8, nz=8, hx=2.0, hy=2.0, hz=2.0, nu=4, nv=40, du=1.0, dv=2.0,
                   sad=100.0, sdd=150.0, n_proj=2)
    p = orc.forward(g, np.ones(g.vol_shape))
    assert np.all(p[:, 0, :] == 0.0) and np.all(p[:, -1, :] == 0.0) and p.max() > 0
    b = orc.back(g, np.ones(g.proj_shape))
    assert b.min() == 0.0 and b.max() > 0


# ---------------------------------------------------------------------------
# NEXT-1: the paper's Eq. 6 back-projector, oracle_back_eq6
# ---------------------------------------------------------------------------

def test_P15_eq6_isocentre_voxel_and_theta0_by_hand(orc):
    """Values the paper's formulas fix by hand.  (i) A voxel at the isocentre sees u* = v* = 0, l = SAD, L = L0 in
    every view (A6, L401-L406), so with T = 1 Eq. 6 gives  dV/(du dv) * N_theta * L0^2 / SAD^2.  (ii) At theta = 0
    the appendix formulas hold literally (A6: u* = -(y-ys) L0/(x-xs), v* = (z-zs) L0/(x-xs); A2: L^2 = L0^2+u^2+v^2);
    a T that is linear in (u, v) is reproduced exactly by bilinear interpolation, so the expected value needs no
    interpolation code."""
    g = I.Geometry(nx=5, ny=5, nz=5, hx=2.0, hy=2.0, hz=3.0, nu=64, nv=64, du=1.5, dv=2.5, sad=400.0, sdd=700.0,
                   n_proj=7, angles=np.deg2rad([0.0, 31.0, 77.0, 140.0, 201.0, 260.0, 333.0]))
    b = orc.back_eq6(g, np.ones(g.proj_shape))
    assert b[2, 2, 2] == pytest.approx(2.0 * 2.0 * 3.0 / (1.5 * 2.5) * 7 * 700.0 ** 2 / 400.0 ** 2, rel=1e-12)
    g0 = g.replace(n_proj=1, angles=np.array([0.0]))
    u = (np.arange(g0.nu) - (g0.nu - 1) / 2) * g0.du
    v = (np.arange(g0.nv) - (g0.nv - 1) / 2) * g0.dv
    U, V = np.meshgrid(u, v)
    a0, a1, a2 = 0.7, 0.013, -0.021
    b = orc.back_eq6(g0, (a0 + a1 * U + a2 * V)[None])
    for (i, j, k) in [(0, 0, 0), (4, 1, 3), (2, 4, 0), (3, 3, 4)]:
        x, y, z = (i - 2) * 2.0, (j - 2) * 2.0, (k - 2) * 3.0
        xs = -400.0
        us, vs = -(y - 0.0) * 700.0 / (x - xs), (z - 0.0) * 700.0 / (x - xs)
        L = np.sqrt(700.0 ** 2 + us ** 2 + vs ** 2)
        l2 = (x - xs) ** 2 + y ** 2 + z ** 2
        want = 12.0 / 3.75 * L ** 3 / (700.0 * l2) * (a0 + a1 * us + a2 * vs)
        assert b[k, j, i] == pytest.approx(want, rel=1e-12), (i, j, k)


def test_P16_eq6_agrees_with_the_exact_transpose_in_the_continuum_limit_and_not_at_config_sampling(orc):
    """Survey S1: with a detector much finer than the voxel footprint and a smooth T, Eq. 6 and the exact transpose
    agree to ~1 %; at the configs' sampling (footprint ~ 1.9 pixels) they differ by tens of per cent voxel by voxel
    (aliasing of the footprint against the pixel grid) -- the two are not interchangeable."""
    Tfun = lambda uu, vv: 1.0 + 0.004 * uu - 0.003 * vv + 1e-5 * uu * vv
    def both(nu, du):
        g = I.Geometry(nx=8, ny=8, nz=8, hx=2.0, hy=2.0, hz=2.0, nu=nu, nv=nu, du=du, dv=du, sad=400.0, sdd=600.0,
                       n_proj=3, angles=np.deg2rad([10.0, 130.0, 250.0]))
        u = (np.arange(nu) - (nu - 1) / 2) * du
        U, V = np.meshgrid(u, u)
        T = np.repeat(Tfun(U, V)[None], 3, axis=0)
        return orc.back(g, T), orc.back_eq6(g, T)
    exact, eq6 = both(400, 0.1)
    assert np.abs(eq6 / exact - 1).max() < 0.02
    exact, eq6 = both(14, 2.9)        # footprint 2 * 1.5 / 2.9 ~ 1 pixel
    assert np.abs(eq6 / exact - 1).max() > 0.05


def test_eq6_taps_outside_the_detector_are_zero(orc):
    """Reading S19: a voxel whose (u*, v*) falls off the detector by more than a pixel gets nothing from that view."""
    g = I.Geometry(nx=9, ny=9, nz=9, hx=4.0, hy=4.0, hz=4.0, nu=6, nv=6, du=1.0, dv=1.0, sad=300.0, sdd=450.0,
                   n_proj=1)
    b = orc.back_eq6(g, np.ones(g.proj_shape))
    assert b[4, 4, 4] > 0 and b[0, 4, 4] == 0.0 and b[4, 0, 4] == 0.0 and b[8, 8, 4] == 0.0


def test_P1_sample_count_equals_brute_force_count(orc):
    """S, the unit of the GUPS metric ("ray-tracing"; reading S2: one (ray, voxel) pair with positive
    length): the traversal's count equals the number of (ray, voxel) pairs whose slab-method length
    (`ray_box_len`, pinned by the hand surds) is positive, on a small off-centre anisotropic grid with generic angles
    (no ray lies in a voxel face: the shortest positive length is far from 0)."""
    g = I.Geometry(nx=9, ny=11, nz=7, hx=1.7, hy=1.3, hz=2.1, nu=10, nv=8, du=2.3, dv=2.9, sad=80.0, sdd=130.0,
                   n_proj=4, vol_off=(0.7, -0.4, 0.3), det_off_u=0.31, det_off_v=-0.17,
                   angles=np.deg2rad([13.0, 101.5, 222.2, 341.0]))
    _, S = orc.forward(g, np.ones(g.vol_shape), return_samples=True)
    h = 0.5 * np.array([g.hx, g.hy, g.hz])
    centres = [np.array([(i - (g.nx - 1) / 2) * g.hx + g.vol_off[0], (j - (g.ny - 1) / 2) * g.hy + g.vol_off[1],
                         (k - (g.nz - 1) / 2) * g.hz + g.vol_off[2]])
               for k in range(g.nz) for j in range(g.ny) for i in range(g.nx)]
    count, shortest, per_ray = 0, np.inf, []
    for a in range(g.n_proj):
        for iv in range(g.nv):
            for iu in range(g.nu):
                S0, D = orc.ray(g, a, iu, iv)
                n = 0
                for c in centres:
                    ln = orc.ray_box_len(S0, D, c - h, c + h)
                    if ln > 0.0:
                        n += 1
                        shortest = min(shortest, ln)
                per_ray.append(n)
                count += n
    assert shortest > 1e-6                      # no grazing pair decides the count
    assert S == count == 3882
    assert max(per_ray) <= g.nx + g.ny + g.nz   # a ray crosses at most nx + ny + nz - 2 voxels
