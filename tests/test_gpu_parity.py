"""Parity of the CUDA path (through the C ABI of include/cbct.h) against the CPU oracle, element
by element on the same seeded inputs.  Tolerances (BASELINE.json north_star):
    P, P^T        relative L2 <= 1e-5 (per projection / per volume)
    adjoint       |<Pf,g> - <f,P^T g>| <= 1e-5 |<Pf,g>|
    TV-prox       output relative L2 <= 1e-5, identical inner-iteration and trial counts
    transfers     relative L2 <= 1e-6
    FBS volume    relative L2 <= 1e-3 after the fixed iteration count
    run-to-run    bitwise identical
"""
import numpy as np
import pytest

from paper_1001_0599_b200 import inputs as I

pytestmark = pytest.mark.gpu

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
    n = np.linalg.norm(b)
    return np.linalg.norm(a - b) / n if n > 0 else np.linalg.norm(a)


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


# geometries spanning several tiles and ragged tails of every kernel's block shape
def geoms():
    out = {}
    out["config1"] = I.config(1).geom
    # odd sizes, anisotropic voxels, off-centre volume and detector, irregular angles
    out["ragged"] = I.Geometry(nx=37, ny=45, nz=19, hx=1.7, hy=1.3, hz=2.9, nu=67, nv=41, du=1.9, dv=2.3,
                               sad=400.0, sdd=650.0, n_proj=7, vol_off=(3.1, -2.2, 1.4), det_off_u=2.5,
                               det_off_v=-1.7, angles=np.deg2rad([0.0, 45.0, 90.0, 133.3, 180.0, 270.0, 311.1]))
    # config-4-like anisotropy (0.5 x 0.5 x 1 mm) at reduced size, wide detector -> truncation in v
    out["aniso"] = I.Geometry(nx=96, ny=96, nz=40, hx=0.5, hy=0.5, hz=1.0, nu=128, nv=48, du=0.776, dv=0.776,
                              sad=1000.0, sdd=1500.0, n_proj=12)
    # 64^3 at config-2 sampling, 9 views
    out["cube64"] = I.Geometry(nx=64, ny=64, nz=64, hx=2.0, hy=2.0, hz=2.0, nu=128, nv=96, du=1.55, dv=1.55,
                               sad=1000.0, sdd=1500.0, n_proj=9)
    # quarter-turn symmetric (square centred in-plane grid, 16 views), odd nz / nv, off-centre in z and v
    out["sym48"] = I.Geometry(nx=48, ny=48, nz=21, hx=1.5, hy=1.5, hz=2.0, nu=80, nv=37, du=1.4, dv=1.7,
                              sad=600.0, sdd=900.0, n_proj=16, vol_off=(0.0, 0.0, 1.3), det_off_u=0.9,
                              det_off_v=-2.1,
                              angles=np.deg2rad(11.0) + 2 * np.pi * np.arange(16) / 16)
    # coarse voxels on a fine detector: a voxel's shadow is ~9 columns wide, which takes the back-projector's
    # general kernel (back_kernel) instead of the shared-memory list kernel (at most 5 columns per voxel and view)
    out["wide"] = I.Geometry(nx=24, ny=20, nz=12, hx=4.0, hy=4.0, hz=4.0, nu=160, nv=96, du=1.0, dv=1.0,
                             sad=500.0, sdd=800.0, n_proj=5, angles=np.deg2rad([3.0, 80.0, 155.0, 222.0, 301.0]))
    # the same regime with every symmetry on (square centred grid, 8 equally spaced views)
    out["wide8"] = I.Geometry(nx=24, ny=24, nz=12, hx=4.0, hy=4.0, hz=4.0, nu=160, nv=96, du=1.0, dv=1.0,
                              sad=500.0, sdd=800.0, n_proj=8)
    return out


GEOMS = geoms()
# every geometry through the generic kernels; the symmetric ones also through the quarter-turn kernels
CASES = [(n, True) for n in GEOMS] + [(n, False) for n in ("config1", "aniso", "sym48", "wide8")]


@pytest.mark.parametrize("name,generic", CASES)
def test_forward_projector_matches_oracle(torch, cbct, orc, name, generic):
    g = GEOMS[name]
    f = I.uniform_volume(g, 11)
    want = orc.forward(g, f)
    with cbct.geometry_create(g, no_symmetry=generic) as h:
        assert h.symmetry == (1 if generic else {"config1": 8, "aniso": 8, "sym48": 4, "cube64": 2, "wide8": 8}.get(name, 1))
        p = torch.empty(g.proj_shape, device="cuda", dtype=torch.float32)
        h.forward_project(dev(torch, f), p)
        got = p.cpu().numpy()
    assert want.max() > 0
    for a in range(g.n_proj):
        assert rel_l2(got[a], want[a]) <= TOL_PROJ, (name, a, rel_l2(got[a], want[a]))
    # rays that miss the volume are exactly zero on both sides
    assert np.array_equal(got == 0.0, want == 0.0) or np.abs(got[want == 0.0]).max() < 1e-6


@pytest.mark.parametrize("name,generic", CASES)
def test_back_projector_matches_oracle(torch, cbct, orc, name, generic):
    g = GEOMS[name]
    q = I.uniform_projections(g, 12)
    want = orc.back(g, q)
    with cbct.geometry_create(g, no_symmetry=generic) as h:
        b = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
        h.back_project(dev(torch, q), b)
        got = b.cpu().numpy()
    assert rel_l2(got, want) <= TOL_PROJ, (name, rel_l2(got, want))
    # worst voxel, relative to the volume's scale (not just the L2 average)
    assert np.abs(got - want).max() <= 1e-4 * np.abs(want).max()


@pytest.mark.parametrize("name,generic", CASES)
def test_adjoint_identity_on_device(torch, cbct, name, generic):
    """<P f, q> = <f, P^T q> to 1e-5 relative (north_star), dot products in fp64 on the host."""
    g = GEOMS[name]
    f = I.uniform_volume(g, 21)
    q = I.uniform_projections(g, 22) - 0.3
    with cbct.geometry_create(g, no_symmetry=generic) as h:
        p = torch.empty(g.proj_shape, device="cuda", dtype=torch.float32)
        b = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
        h.forward_project(dev(torch, f), p)
        h.back_project(dev(torch, q), b)
        lhs = np.vdot(p.cpu().numpy().astype(np.float64), q.astype(np.float64))
        rhs = np.vdot(f.astype(np.float64), b.cpu().numpy().astype(np.float64))
    assert abs(lhs - rhs) <= 1e-5 * abs(lhs), (lhs, rhs)


def test_forward_projector_view_pairs_agree_with_base_views(torch, cbct, orc):
    """Where the view set is also symmetric under theta -> -theta the forward projector walks view PAIRS (16 rays per weight:
    quarter turns x reflection x z-mirror); CBCT_KERNEL_NO_REFLECTION keeps it on base views.  Same projections to fp32
    rounding, both within 1e-5 of the oracle -- with an even and an odd number of base views (the middle view of an even
    count is its own partner and walks half its columns), and with the reflection refused (detector off-centre in u)."""
    cases = {"even": I.Geometry(nx=40, ny=40, nz=18, hx=1.5, hy=1.5, hz=2.0, nu=72, nv=30, du=1.3, dv=1.6, sad=600.0, sdd=900.0,
                                n_proj=16),
             "odd": I.Geometry(nx=40, ny=40, nz=18, hx=1.5, hy=1.5, hz=2.0, nu=72, nv=30, du=1.3, dv=1.6, sad=600.0, sdd=900.0,
                               n_proj=12),
             "config1": GEOMS["config1"]}
    for name, g in cases.items():
        f = I.uniform_volume(g, 17)
        want = orc.forward(g, f)
        outs = {}
        for no_refl in (False, True):
            with cbct.geometry_create(g, no_reflection=no_refl) as h:
                assert h.symmetry == 8
                p = torch.empty(g.proj_shape, device="cuda", dtype=torch.float32)
                h.forward_project(dev(torch, f), p)
                outs[no_refl] = p.cpu().numpy()
                assert h.shard_units(0)[0] == ((g.n_proj // 4) if no_refl else (g.n_proj // 4) // 2 + 1), name
        for a in range(g.n_proj):
            for o in outs.values():
                assert rel_l2(o[a], want[a]) <= TOL_PROJ, (name, a)
        assert rel_l2(outs[False], outs[True]) <= 1e-6
    g = cases["even"].replace(det_off_u=0.4)
    with cbct.geometry_create(g) as h:
        assert h.shard_units(0)[0] == g.n_proj // 4            # no pairing with the detector off-centre


def test_forward_projector_folded_copy_agrees_with_per_image_cells(torch, cbct, orc):
    """Quarter-turn + mirror symmetric levels read the staged copy FOLDED onto the first quadrant (one 32-byte entry = a cell's
    four quarter-turn images and their z-mirrors; the sums are kept in the frame of the walk's current quadrant and turned when
    it changes); CBCT_KERNEL_NO_FOLD keeps one 8-byte cell per image.  Same weights: projections equal to fp32 rounding
    -- with and without view pairs, with an odd and an even number of base views, on a grid whose rays cross the centre plane of
    the minor axis at every slope (all views of a full turn), with a detector that looks past the volume (rows and columns that
    miss it, rays that leave through the top), and within 1e-5 of the oracle."""
    cases = {"even": I.Geometry(nx=40, ny=40, nz=18, hx=1.5, hy=1.5, hz=2.0, nu=72, nv=30, du=1.3, dv=1.6, sad=600.0, sdd=900.0,
                                n_proj=16),
             "odd": I.Geometry(nx=40, ny=40, nz=18, hx=1.5, hy=1.5, hz=2.0, nu=72, nv=30, du=1.3, dv=1.6, sad=600.0, sdd=900.0,
                               n_proj=12),
             "wide": I.Geometry(nx=24, ny=24, nz=40, hx=2.0, hy=2.0, hz=1.0, nu=96, nv=64, du=1.5, dv=1.5, sad=300.0, sdd=500.0,
                                n_proj=20),
             # quarter turns without the reflection (first view off 0 degrees): the folded walk of 8 rays
             "turned": I.Geometry(nx=40, ny=40, nz=18, hx=1.5, hy=1.5, hz=2.0, nu=72, nv=30, du=1.3, dv=1.6, sad=600.0, sdd=900.0,
                                  n_proj=16, angles=np.deg2rad(11.0) + 2 * np.pi * np.arange(16) / 16),
             # a first quadrant of 18 x 18 cells: staging tiles with ragged edges on both in-plane axes
             "n36": I.Geometry(nx=36, ny=36, nz=14, hx=1.5, hy=1.5, hz=2.0, nu=64, nv=24, du=1.3, dv=1.6, sad=600.0, sdd=900.0,
                               n_proj=8),
             "config1": GEOMS["config1"], "aniso": GEOMS["aniso"], "wide8": GEOMS["wide8"]}
    for name, g in cases.items():
        f = I.uniform_volume(g, 23)
        want = orc.forward(g, f)
        for no_refl in (False, True):
            outs = {}
            for no_fold in (False, True):
                with cbct.geometry_create(g, no_reflection=no_refl, no_fold=no_fold) as h:
                    assert h.symmetry == 8, name
                    p = torch.empty(g.proj_shape, device="cuda", dtype=torch.float32)
                    h.forward_project(dev(torch, f), p)
                    outs[no_fold] = p.cpu().numpy()
            for a in range(g.n_proj):
                assert rel_l2(outs[False][a], want[a]) <= TOL_PROJ, (name, no_refl, a)
            # same weights; the z-neighbour cells of slabs without an in-plane crossing are added in batches (another order of the
            # same terms): equal to fp32 rounding
            assert rel_l2(outs[False], outs[True]) <= 1e-6, (name, no_refl, rel_l2(outs[False], outs[True]))
            if no_refl:     # the 8-ray walk adds every term in forward_kernel's order: the same bits
                assert outs[False].tobytes() == outs[True].tobytes(), (name, float(np.abs(outs[False] - outs[True]).max()))


@pytest.mark.parametrize("name", ["ragged", "sym48"])
def test_projectors_are_bitwise_deterministic(torch, cbct, name):
    g = GEOMS[name]
    f, q = dev(torch, I.uniform_volume(g, 31)), dev(torch, I.uniform_projections(g, 32))
    outs = []
    for _ in range(2):
        with cbct.geometry_create(g) as h:
            p = torch.empty(g.proj_shape, device="cuda", dtype=torch.float32)
            b = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
            h.forward_project(f, p)
            h.back_project(q, b)
            outs.append((p.cpu().numpy().tobytes(), b.cpu().numpy().tobytes()))
    assert outs[0] == outs[1]


def test_sample_count_matches_oracle(torch, cbct, orc):
    """S = number of (ray, voxel) pairs with positive length: the unit of the GUPS metric."""
    for name in ("config1", "ragged"):
        g = GEOMS[name]
        _, S = orc.forward(g, np.ones(g.vol_shape), return_samples=True)
        with cbct.geometry_create(g) as h:
            got = h.count_samples()
        # pairs whose length is within rounding of zero (a ray through a voxel edge or corner; common on
        # config 1's centred, symmetric grid) are counted by one side and not the other
        assert abs(got - S) <= 2e-3 * S, (name, got, S)


def test_edge_cases_missing_rays_and_unseen_voxels(torch, cbct, orc):
    """Detector far taller than the volume's shadow: rows that miss give 0; unseen voxels give 0."""
    g = I.Geometry(nx=8, ny=8, nz=8, hx=2.0, hy=2.0, hz=2.0, nu=4, nv=40, du=1.0, dv=2.0, sad=100.0, sdd=150.0,
                   n_proj=2)
    with cbct.geometry_create(g) as h:
        p = torch.full(g.proj_shape, 7.0, device="cuda", dtype=torch.float32)
        h.forward_project(dev(torch, np.ones(g.vol_shape)), p)
        b = torch.full(g.vol_shape, 7.0, device="cuda", dtype=torch.float32)
        h.back_project(dev(torch, np.ones(g.proj_shape)), b)
    p, b = p.cpu().numpy(), b.cpu().numpy()
    assert np.all(p[:, 0, :] == 0.0) and np.all(p[:, -1, :] == 0.0) and p.max() > 0
    want = orc.back(g, np.ones(g.proj_shape))
    assert rel_l2(b, want) <= TOL_PROJ and np.all(b[want == 0.0] == 0.0)
    # single voxel, single pixel, single view
    g1 = I.Geometry(nx=1, ny=1, nz=1, hx=3.0, hy=3.0, hz=3.0, nu=1, nv=1, du=1.0, dv=1.0, sad=100.0, sdd=150.0,
                    n_proj=1, det_off_u=0.2, det_off_v=0.1)
    with cbct.geometry_create(g1) as h:
        p = torch.empty(g1.proj_shape, device="cuda", dtype=torch.float32)
        h.forward_project(dev(torch, np.full(g1.vol_shape, 2.0)), p)
    assert p.item() == pytest.approx(orc.forward(g1, np.full(g1.vol_shape, 2.0)).item(), rel=1e-6)


@pytest.mark.parametrize("host_armijo", [False, True])
@pytest.mark.parametrize("bc", [(I.BC_ZERO, I.BC_REFLECT), (I.BC_REFLECT, I.BC_REFLECT), (I.BC_ZERO, I.BC_ZERO)])
@pytest.mark.parametrize("shape", [(37, 45, 19), (132, 21, 11), (256, 16, 5)])
def test_tv_energy_and_prox_match_oracle(torch, cbct, orc, bc, host_armijo, shape):
    """Both control paths of the Armijo loop: the cooperative kernel that decides on the device (default) and the
    host-sequenced loop (CBCT_KERNEL_HOST_ARMIJO).  Shapes: the 32-voxel warp tiles (nx = 37: ragged in x, y and z), and
    the 16-byte tiles of tv.cu (nx % 4 == 0, nx >= 128): 132 x 21 x 11 has a second tile column with ONE valid lane (so the
    p_x column left of a tile and the right-neighbour column are both exercised), ragged rows and two z-chunks;
    256 x 16 x 5 fills both tile columns exactly."""
    nx, ny, nz = shape
    g = I.Geometry(nx=nx, ny=ny, nz=nz, hx=1.7, hy=1.3, hz=2.9, nu=8, nv=8, du=2.0, dv=2.0, sad=400.0, sdd=650.0,
                   n_proj=1, bc_xy=bc[0], bc_z=bc[1])
    rng = np.random.default_rng(41)
    base = I.paint([I.Ellipsoid((2.0, -3.0, 1.0), (20.0, 18.0, 16.0), 0.3, 0.02),
                    I.Ellipsoid((-8.0, 5.0, -4.0), (7.0, 9.0, 8.0), 1.0, 0.01)], g)
    gg = (base + 0.002 * rng.standard_normal(g.vol_shape)).astype(np.float32)
    setup = I.FbsSetup(eps_delta=1e-5, max_inner=8, rel_tol=0.0)
    w = 2e-3
    want, wrep = orc.tv_prox(g, gg, w, setup)
    with cbct.geometry_create(g, host_armijo=host_armijo) as h:
        e1 = h.tv_energy(dev(torch, gg), setup.eps_delta)
        f = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
        rep = h.tv_prox(dev(torch, gg), f, w, setup)
        got = f.cpu().numpy()
        # with the non-negativity truncation fused into the last write
        f2 = torch.empty_like(f)
        h.tv_prox(dev(torch, gg), f2, w, setup, nonneg=True)
    assert e1 == pytest.approx(orc.tv_energy(g, gg, setup.eps_delta), rel=1e-6)
    assert (rep.inner_iters, rep.trials) == (wrep.inner_iters, wrep.trials)
    assert rep.inner_iters == 8
    assert rep.e_first == pytest.approx(wrep.e_first, rel=1e-6)
    assert rep.e_last == pytest.approx(wrep.e_last, rel=1e-6)
    assert rel_l2(got, want) <= 1e-5
    assert rel_l2(got - gg, want - gg) <= 1e-3          # the update itself, not just f
    assert np.array_equal(f2.cpu().numpy(), np.maximum(got, 0.0))
    assert rep.e_last < rep.e_first


def test_tv_prox_unaligned_volumes_take_the_scalar_tiles(torch, cbct, orc):
    """nx = 128 qualifies for the 16-byte tiles, buffers 4 bytes off a 16-byte boundary do not: same result either way."""
    g = I.Geometry(nx=128, ny=9, nz=6, hx=1.0, hy=1.5, hz=2.0, nu=8, nv=8, du=2.0, dv=2.0, sad=400.0, sdd=650.0,
                   n_proj=1, bc_xy=I.BC_ZERO, bc_z=I.BC_REFLECT)
    rng = np.random.default_rng(43)
    gg = (0.01 + 0.003 * rng.standard_normal(g.vol_shape)).astype(np.float32)
    setup = I.FbsSetup(eps_delta=1e-5, max_inner=3, rel_tol=0.0)
    want, wrep = orc.tv_prox(g, gg, 2e-3, setup)
    n = gg.size
    with cbct.geometry_create(g) as h:
        outs = []
        for off in (0, 1):
            src = torch.zeros(n + 4, device="cuda", dtype=torch.float32)
            dst = torch.zeros(n + 4, device="cuda", dtype=torch.float32)
            gv, fv = src[off:off + n].view(g.vol_shape), dst[off:off + n].view(g.vol_shape)
            gv.copy_(dev(torch, gg))
            rep = h.tv_prox(gv, fv, 2e-3, setup)
            assert (rep.inner_iters, rep.trials) == (wrep.inner_iters, wrep.trials)
            assert h.tv_energy(gv, setup.eps_delta) == pytest.approx(orc.tv_energy(g, gg, setup.eps_delta), rel=1e-6)
            outs.append(fv.cpu().numpy().copy())
    assert rel_l2(outs[0], want) <= 1e-5 and rel_l2(outs[1], want) <= 1e-5
    assert rel_l2(outs[0], outs[1]) <= 1e-6


def test_tv_tile_families_agree(torch, cbct):
    """CBCT_KERNEL_TV_SCALAR_TILES keeps a 16-byte-eligible volume on the 32-voxel tiles: both families give the same
    descent (identical counts, volumes to fp32 rounding of the fp64 sums' inputs) -- zero-BC in-plane, several tile columns
    and rows, more z-chunks than one."""
    g = I.Geometry(nx=260, ny=37, nz=23, hx=0.9, hy=1.1, hz=1.7, nu=8, nv=8, du=2.0, dv=2.0, sad=400.0, sdd=650.0,
                   n_proj=1, bc_xy=I.BC_ZERO, bc_z=I.BC_REFLECT)
    rng = np.random.default_rng(44)
    gg = dev(torch, 0.01 + 0.003 * rng.standard_normal(g.vol_shape))
    setup = I.FbsSetup(eps_delta=1e-5, max_inner=5, rel_tol=0.0)
    outs, reps = [], []
    for scalar in (False, True):
        with cbct.geometry_create(g, tv_scalar_tiles=scalar) as h:
            f = torch.empty_like(gg)
            reps.append(h.tv_prox(gg, f, 3e-3, setup, nonneg=True))
            outs.append(f.cpu().numpy())
    assert (reps[0].inner_iters, reps[0].trials) == (reps[1].inner_iters, reps[1].trials) and reps[0].trials > reps[0].inner_iters
    assert reps[0].e_last == pytest.approx(reps[1].e_last, rel=1e-9)
    assert rel_l2(outs[0], outs[1]) <= 1e-6


@pytest.mark.parametrize("host_armijo", [False, True])
@pytest.mark.parametrize("nx", [16, 128])
def test_tv_prox_degenerate_cases(torch, cbct, host_armijo, nx):
    g = I.Geometry(nx=nx, ny=12, nz=6, hx=1.0, hy=1.0, hz=1.0, nu=8, nv=8, du=2.0, dv=2.0, sad=400.0, sdd=650.0,
                   n_proj=1, bc_xy=I.BC_REFLECT, bc_z=I.BC_REFLECT)
    setup = I.FbsSetup()
    with cbct.geometry_create(g, host_armijo=host_armijo) as h:
        const = torch.full(g.vol_shape, 0.013, device="cuda", dtype=torch.float32)
        # constant volume, all-reflective BC: zero TV (north_star check), prox leaves it alone
        assert h.tv_energy(const, 0.0) == 0.0
        f = torch.empty_like(const)
        h.tv_prox(const, f, 1e-3, setup)
        assert torch.equal(f, const)
        # weight 0: copy (and clip)
        x = dev(torch, np.random.default_rng(5).standard_normal(g.vol_shape))
        rep = h.tv_prox(x, f, 0.0, setup, nonneg=True)
        assert rep.inner_iters == 0 and torch.equal(f, torch.clamp(x, min=0))
        with pytest.raises(cbct.CbctError):
            h.tv_prox(x, x, 1e-3, setup)             # aliasing is refused


def test_grid_transfers_match_oracle(torch, cbct, orc):
    for bc in ((I.BC_ZERO, I.BC_REFLECT), (I.BC_REFLECT, I.BC_ZERO)):
        g = I.Geometry(nx=40, ny=24, nz=12, hx=1.0, hy=1.0, hz=2.0, nu=36, nv=20, du=2.0, dv=2.0, sad=400.0,
                       sdd=650.0, n_proj=3, bc_xy=bc[0], bc_z=bc[1])
        rng = np.random.default_rng(51)
        fine = rng.random(g.vol_shape).astype(np.float32)
        proj = rng.random(g.proj_shape).astype(np.float32)
        with cbct.geometry_create(g, max_levels=2) as h:
            c = torch.empty(h.vol_shape(1), device="cuda", dtype=torch.float32)
            h.restrict_volume(dev(torch, fine), c)
            pb = torch.empty(h.proj_shape(1), device="cuda", dtype=torch.float32)
            h.bin_projections(dev(torch, proj), pb)
            up = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
            coarse = rng.random(h.vol_shape(1)).astype(np.float32)
            h.prolong_volume(dev(torch, coarse), up)
        assert rel_l2(c.cpu().numpy(), orc.restrict(fine)) <= 1e-6
        assert rel_l2(pb.cpu().numpy(), orc.bin2(proj)) <= 1e-6
        assert rel_l2(up.cpu().numpy(), orc.prolong(coarse, bc[0], bc[1])) <= 1e-6


def test_step_bound_matches_oracle(torch, cbct, orc):
    g = GEOMS["config1"]
    with cbct.geometry_create(g) as h:
        assert h.step_bound() == pytest.approx(orc.step_bound(g), rel=1e-5)


def test_fbs_config1_matches_oracle(torch, cbct, orc):
    """Config 1 of BASELINE.json as stated: 32^3, 8 views, 48x48, TV weight 0.01, 20 iterations, 1 level."""
    cfg = I.config(1)
    y = I.make_projections(cfg)
    want = orc.fbs(cfg.geom, y, cfg.fbs)
    outs = []
    for _ in range(2):
        with cbct.geometry_create(cfg.geom) as h:
            f = torch.zeros(cfg.geom.vol_shape, device="cuda", dtype=torch.float32)
            rep = h.fbs_reconstruct(dev(torch, y), f, cfg.fbs)
            outs.append(f.cpu().numpy())
    got = outs[0]
    assert rel_l2(got, want.f) <= TOL_VOL, rel_l2(got, want.f)
    assert rep.n_iters_total == 20
    np.testing.assert_allclose(rep.objective, want.objective, rtol=1e-4)
    assert rep.step_abs[0] == pytest.approx(want.step_abs[0], rel=1e-5)
    assert np.all(rep.objective[1:] <= rep.objective[:-1] * (1 + 1e-6))
    assert got.min() >= 0.0
    assert outs[0].tobytes() == outs[1].tobytes()                 # bitwise run-to-run
    # S18: an Armijo / stop decision may flip between fp32 and fp64 only at a tie; none of this case's is one
    assert (rep.inner_total, rep.trials_total) == (want.inner_total, want.trials_total)


def test_fbs_multigrid_and_host_entry_match_oracle(torch, cbct, orc):
    """Three levels, noisy data, supplied initial volume, through BOTH entry points."""
    g = I.Geometry(nx=48, ny=48, nz=32, hx=2.0, hy=2.0, hz=2.5, nu=64, nv=48, du=2.4, dv=2.4, sad=1000.0,
                   sdd=1500.0, n_proj=10)
    ell = [I.Ellipsoid((0.0, 0.0, 0.0), (40.0, 34.0, 36.0), 0.0, 0.02)] + \
        I.random_ellipsoids(np.random.default_rng(61), 8, (48.0, 48.0, 40.0), axes_range=(4.0, 14.0))
    y = I.poisson_log(I.analytic_projections(ell, g), 1e5, 62).astype(np.float32)
    setup = I.FbsSetup(iters_per_level=(6, 5, 4))
    want = orc.fbs(g, y, setup)
    with cbct.geometry_create(g, max_levels=3) as h:
        f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        rep = h.fbs_reconstruct(dev(torch, y), f, setup)
        got = f.cpu().numpy()
        host = np.zeros(g.vol_shape, dtype=np.float32)
        h.fbs_reconstruct_host(y, host, setup)
    assert rel_l2(got, want.f) <= TOL_VOL, rel_l2(got, want.f)
    assert host.tobytes() == got.tobytes()
    np.testing.assert_allclose(rep.objective, want.objective, rtol=1e-4)
    np.testing.assert_allclose(rep.step_abs, want.step_abs, rtol=1e-5)
    # with an initial volume (restricted down to the coarsest level first)
    f0 = I.paint(ell, g)
    setup2 = I.FbsSetup(iters_per_level=(2, 2))
    want2 = orc.fbs(g, y, setup2, f0=f0)
    with cbct.geometry_create(g, max_levels=2) as h:
        f = dev(torch, f0)
        h.fbs_reconstruct(dev(torch, y), f, setup2, use_initial=True)
    assert rel_l2(f.cpu().numpy(), want2.f) <= TOL_VOL


def test_fbs_tv_off_is_landweber_on_device(torch, cbct, orc):
    g = GEOMS["config1"]
    y = I.make_projections(I.config(1))
    setup = I.FbsSetup(tv_weight=0.0, step=0.9, iters_per_level=(5,), nonneg=False)
    want = orc.fbs(g, y, setup)
    with cbct.geometry_create(g) as h:
        f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        h.fbs_reconstruct(dev(torch, y), f, setup)
    assert rel_l2(f.cpu().numpy(), want.f) <= 1e-5


def test_error_paths(torch, cbct):
    g = GEOMS["config1"]
    with cbct.geometry_create(g) as h:
        f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        y = torch.zeros(g.proj_shape, device="cuda", dtype=torch.float32)
        with pytest.raises(cbct.CbctError):
            h.fbs_reconstruct(y, f, I.FbsSetup(iters_per_level=(1, 1)))       # 2 levels, 1 provisioned
        with pytest.raises(cbct.CbctError):
            h.fbs_reconstruct(y, f, I.FbsSetup(step=2.5))
        with pytest.raises(ValueError):
            h.forward_project(f[:4], y)
        with pytest.raises((ValueError, cbct.CbctError)):
            h.forward_project(f, y, level=1)                                  # level not provisioned
    # voxels too flat in z for the cone angle: the driving-axis traversal refuses, loudly
    flat = I.Geometry(nx=16, ny=16, nz=64, hx=4.0, hy=4.0, hz=0.05, nu=16, nv=64, du=4.0, dv=4.0, sad=100.0,
                      sdd=150.0, n_proj=4)
    with pytest.raises(cbct.CbctError) as e:
        cbct.geometry_create(flat)
    assert e.value.status == 2


# ---------------------------------------------------------------------------
# NEXT-1: the paper's Eq. 6 back-projector
# ---------------------------------------------------------------------------

@pytest.mark.parametrize("name", list(GEOMS))
def test_eq6_back_projector_matches_oracle(torch, cbct, orc, name):
    g = GEOMS[name]
    q = I.uniform_projections(g, 13)
    want = orc.back_eq6(g, q)
    outs = []
    with cbct.geometry_create(g) as h:
        for _ in range(2):
            b = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
            h.back_project_eq6(dev(torch, q), b)
            outs.append(b.cpu().numpy())
    assert rel_l2(outs[0], want) <= TOL_PROJ, (name, rel_l2(outs[0], want))
    assert np.abs(outs[0] - want).max() <= 1e-4 * np.abs(want).max()
    assert np.array_equal(outs[0] == 0.0, want == 0.0)             # voxels no view sees are exactly 0 on both sides
    assert outs[0].tobytes() == outs[1].tobytes()


def test_fbs_with_the_papers_eq6_gradient_matches_oracle(torch, cbct, orc):
    """Algorithm A1 as the paper ran it: step 1 with Eq. 6 in place of P^T (an unmatched pair), two levels."""
    g = I.Geometry(nx=48, ny=48, nz=32, hx=2.0, hy=2.0, hz=2.5, nu=64, nv=48, du=2.4, dv=2.4, sad=1000.0,
                   sdd=1500.0, n_proj=10)
    ell = [I.Ellipsoid((0.0, 0.0, 0.0), (40.0, 34.0, 36.0), 0.0, 0.02)] + \
        I.random_ellipsoids(np.random.default_rng(71), 6, (48.0, 48.0, 40.0), axes_range=(4.0, 14.0))
    y = I.poisson_log(I.analytic_projections(ell, g), 1e5, 72).astype(np.float32)
    setup = I.FbsSetup(iters_per_level=(5, 4), backprojector=1, step=0.8)
    want = orc.fbs(g, y, setup)
    with cbct.geometry_create(g, max_levels=2) as h:
        f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        rep = h.fbs_reconstruct(dev(torch, y), f, setup)
        got = f.cpu().numpy()
    assert rel_l2(got, want.f) <= TOL_VOL, rel_l2(got, want.f)
    np.testing.assert_allclose(rep.objective, want.objective, rtol=1e-4)
    # and it is a different iteration from the matched pair's
    exact = orc.fbs(g, y, I.FbsSetup(iters_per_level=(5, 4), step=0.8))
    assert rel_l2(want.f, exact.f) > 1e-3


def test_fbs_convergence_stopping_matches_oracle(torch, cbct, orc):
    """NEXT-2: 'until convergence' with the relative-change test, two levels; same iteration counts, same volume."""
    g = I.Geometry(nx=48, ny=48, nz=32, hx=2.0, hy=2.0, hz=2.5, nu=64, nv=48, du=2.4, dv=2.4, sad=1000.0,
                   sdd=1500.0, n_proj=10)
    ell = [I.Ellipsoid((0.0, 0.0, 0.0), (40.0, 34.0, 36.0), 0.0, 0.02)] + \
        I.random_ellipsoids(np.random.default_rng(91), 6, (48.0, 48.0, 40.0), axes_range=(4.0, 14.0))
    y = I.poisson_log(I.analytic_projections(ell, g), 1e5, 92).astype(np.float32)
    setup = I.FbsSetup(iters_per_level=(30, 30), conv_tol=0.03)
    want = orc.fbs(g, y, setup)
    with cbct.geometry_create(g, max_levels=2) as h:
        f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        rep = h.fbs_reconstruct(dev(torch, y), f, setup)
        got = f.cpu().numpy()
    assert rep.iters_done == want.iters_done and all(0 < n < 30 for n in rep.iters_done)
    assert rep.n_iters_total == sum(want.iters_done) and len(rep.objective) == len(want.objective)
    assert rel_l2(got, want.f) <= TOL_VOL
    np.testing.assert_allclose(rep.objective, want.objective, rtol=1e-4)


@pytest.mark.parametrize("tv_weight", [0.01, 300.0])
def test_fbs_look_ahead_projection_changes_nothing(torch, cbct, orc, tv_weight):
    """Without the objective monitor the driver queues the next iteration's forward projection behind the first TV
    trial pass (whose volume is the result when that step is accepted and last) and redoes it otherwise.  Both ways
    must give bit for bit the volume of the plain sequence (objective monitor on: no look-ahead).  tv_weight 0.01:
    every prox call ends after one step (look-ahead used); 300: several descent steps per call (look-ahead redone)."""
    g = I.Geometry(nx=48, ny=48, nz=32, hx=2.0, hy=2.0, hz=2.5, nu=64, nv=48, du=2.4, dv=2.4, sad=1000.0,
                   sdd=1500.0, n_proj=12)
    ell = [I.Ellipsoid((0.0, 0.0, 0.0), (40.0, 34.0, 36.0), 0.0, 0.02)] + \
        I.random_ellipsoids(np.random.default_rng(101), 6, (48.0, 48.0, 40.0), axes_range=(4.0, 14.0))
    y = I.poisson_log(I.analytic_projections(ell, g), 1e5, 102).astype(np.float32)
    setup = I.FbsSetup(iters_per_level=(4, 6), tv_weight=tv_weight)
    outs, reps = [], []
    with cbct.geometry_create(g, max_levels=2, host_armijo=True) as h:
        for objective in (True, False, False):
            f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
            reps.append(h.fbs_reconstruct(dev(torch, y), f, setup, objective=objective))
            outs.append(f.cpu().numpy())
    assert outs[0].tobytes() == outs[1].tobytes() == outs[2].tobytes()
    assert reps[0].inner_total == reps[1].inner_total and reps[0].trials_total == reps[1].trials_total
    assert (reps[0].inner_total > 10) == (tv_weight > 1.0)           # the two regimes the test is about
    want = orc.fbs(g, y, setup)
    assert rel_l2(outs[1], want.f) <= TOL_VOL


def _noisy_48():
    g = I.Geometry(nx=48, ny=48, nz=32, hx=2.0, hy=2.0, hz=2.5, nu=64, nv=48, du=2.4, dv=2.4, sad=1000.0,
                   sdd=1500.0, n_proj=12)
    ell = [I.Ellipsoid((0.0, 0.0, 0.0), (40.0, 34.0, 36.0), 0.0, 0.02)] + \
        I.random_ellipsoids(np.random.default_rng(111), 6, (48.0, 48.0, 40.0), axes_range=(4.0, 14.0))
    return g, I.poisson_log(I.analytic_projections(ell, g), 1e5, 112).astype(np.float32)


def test_fbs_look_ahead_backtracked_and_last(torch, cbct, orc):
    """The look-ahead projection is queued behind the FIRST trial of a prox call; when that trial is rejected and a
    shrunken step is accepted AND is the last (max_inner = 1), the queued projection saw a rejected volume and must be
    redone.  Bitwise equality with the plain sequence (objective monitor on), and parity with the oracle."""
    g, y = _noisy_48()
    setup = I.FbsSetup(iters_per_level=(3, 5), tv_weight=3000.0, max_inner=1)
    outs, reps = [], []
    with cbct.geometry_create(g, max_levels=2, host_armijo=True) as h:
        for objective in (True, False, False):
            f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
            reps.append(h.fbs_reconstruct(dev(torch, y), f, setup, objective=objective))
            outs.append(f.cpu().numpy())
    assert reps[1].trials_total > reps[1].inner_total          # some accepted step had been backtracked to
    assert reps[1].inner_total == 8                             # one descent step per prox call
    assert outs[0].tobytes() == outs[1].tobytes() == outs[2].tobytes()
    want = orc.fbs(g, y, setup)
    assert (reps[1].inner_total, reps[1].trials_total) == (want.inner_total, want.trials_total)
    assert rel_l2(outs[1], want.f) <= TOL_VOL


@pytest.mark.parametrize("host_armijo", [False, True])
@pytest.mark.parametrize("objective", [True, False])
@pytest.mark.parametrize("kw", [dict(max_inner=1, tv_weight=300.0), dict(max_backtracks=0, tv_weight=3000.0),
                                dict(max_backtracks=1, tv_weight=3000.0)])
def test_fbs_short_prox_budgets_match_oracle(torch, cbct, orc, kw, objective, host_armijo):
    """The ROF sub-solver cut short inside the FBS driver: a single descent step per call, and a backtracking budget
    that runs out (the prox call then keeps f = g: PAPER.md:L155-L159, reading S8) -- with and without the monitor."""
    g, y = _noisy_48()
    setup = I.FbsSetup(iters_per_level=(3, 4), **kw)
    want = orc.fbs(g, y, setup)
    with cbct.geometry_create(g, max_levels=2, host_armijo=host_armijo) as h:
        f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        rep = h.fbs_reconstruct(dev(torch, y), f, setup, objective=objective)
        got = f.cpu().numpy()
    assert (rep.inner_total, rep.trials_total) == (want.inner_total, want.trials_total)
    if "max_backtracks" in kw and kw["max_backtracks"] == 0:
        assert rep.trials_total > rep.inner_total               # the budget did run out in some call
    assert rel_l2(got, want.f) <= TOL_VOL, rel_l2(got, want.f)
    if objective:
        np.testing.assert_allclose(rep.objective, want.objective, rtol=1e-4)


# ---------------------------------------------------------------------------
# NEXT-2: the paper's 4-level schedule and its short-arc / subset acquisition protocols through the whole driver
# ---------------------------------------------------------------------------

def test_fbs_four_level_schedule_matches_oracle(torch, cbct, orc):
    """The paper's driver Omega_8h -> Omega_4h -> Omega_2h -> Omega_h: 64^3 finest, 8^3 coarsest."""
    g = I.Geometry(nx=64, ny=64, nz=64, hx=2.0, hy=2.0, hz=2.0, nu=128, nv=96, du=1.55, dv=1.55, sad=1000.0,
                   sdd=1500.0, n_proj=16)
    ell = [I.Ellipsoid((0.0, 0.0, 0.0), (52.0, 44.0, 50.0), 0.0, 0.02)] + \
        I.random_ellipsoids(np.random.default_rng(121), 8, (64.0, 64.0, 64.0), axes_range=(5.0, 18.0))
    y = I.poisson_log(I.analytic_projections(ell, g), 1e5, 122).astype(np.float32)
    setup = I.FbsSetup(iters_per_level=(5, 4, 3, 2))
    want = orc.fbs(g, y, setup)
    with cbct.geometry_create(g, max_levels=4) as h:
        f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        rep = h.fbs_reconstruct(dev(torch, y), f, setup)
        got = f.cpu().numpy()
        assert h.bound_violations() == 0
    assert rep.n_iters_total == 14 and rep.iters_done == (5, 4, 3, 2)
    assert rel_l2(got, want.f) <= TOL_VOL, rel_l2(got, want.f)
    np.testing.assert_allclose(rep.objective, want.objective, rtol=1e-4)
    np.testing.assert_allclose(rep.step_abs, want.step_abs, rtol=1e-5)
    assert (rep.inner_total, rep.trials_total) == (want.inner_total, want.trials_total)


def _arc_angles(kind):
    if kind == "arc200":            # 40 equally spaced views over a 200 degree arc
        return np.deg2rad(200.0) * np.arange(40) / 40
    # the paper's patient / CatPhan protocol: 40 of 363 projections acquired over 200 degrees (L295, L323);
    # 363 / 40 is not an integer, so the subset is not equally spaced
    idx = np.round(np.arange(40) * 363 / 40).astype(int)
    return (np.deg2rad(200.0) * np.arange(363) / 363)[idx]


@pytest.mark.parametrize("kind", ["arc200", "subset363"])
def test_fbs_short_arc_protocols_match_oracle(torch, cbct, orc, kind):
    """Short-arc acquisitions switch the quarter-turn symmetry off (no view has its three quarter-turn partners) and
    keep the mirror symmetry: the nsym = 1, nmir = 2 kernels through a 2-level reconstruction of noisy data."""
    ang = _arc_angles(kind)
    if kind == "subset363":
        assert len(set(np.round(np.diff(ang), 9))) > 1
    g = I.Geometry(nx=48, ny=48, nz=32, hx=2.0, hy=2.0, hz=2.5, nu=64, nv=48, du=2.4, dv=2.4, sad=1000.0,
                   sdd=1500.0, n_proj=40, angles=ang)
    ell = [I.Ellipsoid((0.0, 0.0, 0.0), (40.0, 34.0, 36.0), 0.0, 0.02)] + \
        I.random_ellipsoids(np.random.default_rng(131), 6, (48.0, 48.0, 40.0), axes_range=(4.0, 14.0))
    y = I.poisson_log(I.analytic_projections(ell, g), 1e5, 132).astype(np.float32)
    setup = I.FbsSetup(iters_per_level=(6, 5))
    want = orc.fbs(g, y, setup)
    with cbct.geometry_create(g, max_levels=2) as h:
        assert h.symmetry == 2 and h.back_path(0) in ("list", "gather")
        f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        rep = h.fbs_reconstruct(dev(torch, y), f, setup)
        got = f.cpu().numpy()
        f.zero_()
        h.fbs_reconstruct(dev(torch, y), f, setup)
        assert f.cpu().numpy().tobytes() == got.tobytes()
    assert rel_l2(got, want.f) <= TOL_VOL, rel_l2(got, want.f)
    np.testing.assert_allclose(rep.objective, want.objective, rtol=1e-4)
    assert (rep.inner_total, rep.trials_total) == (want.inner_total, want.trials_total)


def test_back_projector_paths_agree(torch, cbct, orc):
    """The TMA / shared-memory back-projector and the list kernel it replaces, on the same handle geometry
    (cbct_geometry_desc::kernel_flags): both within 1e-5 of the oracle, within 1e-6 of each other, no tile bound of the
    TMA plan violated -- on config 1, an anisotropic grid, and a ragged one (sizes that are not multiples of the brick)."""
    cases = {"config1": GEOMS["config1"], "aniso": GEOMS["aniso"].replace(hx=1.0, hy=1.0),
             "ragged_sym": I.Geometry(nx=44, ny=44, nz=38, hx=1.5, hy=1.5, hz=1.5, nu=96, nv=70, du=1.1, dv=1.1,
                                      sad=600.0, sdd=900.0, n_proj=12)}
    for name, g in cases.items():
        q = I.uniform_projections(g, 14)
        want = orc.back(g, q)
        outs = {}
        for no_tma in (False, True):
            with cbct.geometry_create(g, no_tma=no_tma) as h:
                assert h.back_path(0) == ("list" if no_tma else "tma"), (name, h.back_path(0))
                b = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
                h.back_project(dev(torch, q), b)
                first = b.cpu().numpy()
                h.back_project(dev(torch, q), b)
                assert b.cpu().numpy().tobytes() == first.tobytes()
                assert h.bound_violations() == 0
                outs[no_tma] = first
        for o in outs.values():
            assert rel_l2(o, want) <= TOL_PROJ, (name, rel_l2(o, want))
            assert np.abs(o - want).max() <= 1e-4 * np.abs(want).max()
        assert rel_l2(outs[False], outs[True]) <= 1e-6
        # the TMA kernel fed by the in-plane list and stage-header tables made at create (the default) and the same kernel
        # working both out itself (CBCT_KERNEL_BACK_LISTS_ON_THE_FLY): one definition of every entry, so the same bits
        with cbct.geometry_create(g, back_lists_on_the_fly=True) as h:
            assert h.back_path(0) == "tma"
            b = torch.empty(g.vol_shape, device="cuda", dtype=torch.float32)
            h.back_project(dev(torch, q), b)
            assert h.bound_violations() == 0
            assert b.cpu().numpy().tobytes() == outs[False].tobytes(), name


def test_fbs_device_and_host_armijo_agree_bitwise(torch, cbct, orc):
    """The cooperative TV-prox kernel (every accept / shrink / stop decision taken on the device) against the
    host-sequenced loop: the same passes in the same order, so the same volume bit for bit and the same counts --
    in the regime of one descent step per call and in the regime of many backtracked steps."""
    g, y = _noisy_48()
    for tv_weight in (0.01, 300.0):
        setup = I.FbsSetup(iters_per_level=(4, 5), tv_weight=tv_weight)
        outs, reps = [], []
        for host in (False, True):
            with cbct.geometry_create(g, max_levels=2, host_armijo=host) as h:
                f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
                reps.append(h.fbs_reconstruct(dev(torch, y), f, setup, objective=False))
                outs.append(f.cpu().numpy())
        assert outs[0].tobytes() == outs[1].tobytes()
        assert (reps[0].inner_total, reps[0].trials_total) == (reps[1].inner_total, reps[1].trials_total)
        assert (reps[0].trials_total > reps[0].inner_total) == (tv_weight > 1.0)
