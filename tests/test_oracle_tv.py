"""Pins of the oracle's TV / ROF pieces and grid transfers."""
import itertools

import numpy as np
import pytest

from paper_1001_0599_b200 import inputs as I

BCS = list(itertools.product([I.BC_ZERO, I.BC_REFLECT], repeat=2))


def vol_geom(n=(7, 6, 5), h=(1.0, 1.5, 2.0), bc_xy=I.BC_ZERO, bc_z=I.BC_REFLECT):
    return I.Geometry(nx=n[0], ny=n[1], nz=n[2], hx=h[0], hy=h[1], hz=h[2], nu=4, nv=4, du=1.0,
                      dv=1.0, n_proj=1, bc_xy=bc_xy, bc_z=bc_z)


def numpy_grad(f, g):
    """Forward differences with the boundary rules of PAPER.md:L161, written with numpy
    padding (independent of the C loops)."""
    def pad(axis, bc):
        if bc == I.BC_ZERO:
            return np.concatenate([f, np.zeros_like(np.take(f, [0], axis))], axis)
        return np.concatenate([f, np.take(f, [-1], axis)], axis)
    gx = np.diff(pad(2, g.bc_xy), axis=2) / g.hx
    gy = np.diff(pad(1, g.bc_xy), axis=1) / g.hy
    gz = np.diff(pad(0, g.bc_z), axis=0) / g.hz
    return gx, gy, gz


@pytest.mark.parametrize("bc_xy,bc_z", BCS)
def test_tv_energy_matches_numpy_definition(orc, bc_xy, bc_z):
    g = vol_geom(bc_xy=bc_xy, bc_z=bc_z)
    f = np.random.default_rng(0).random(g.vol_shape)
    gx, gy, gz = numpy_grad(f, g)
    for delta in (0.0, 1e-3, 0.5):
        want = np.sqrt(gx ** 2 + gy ** 2 + gz ** 2 + delta ** 2).mean()
        assert orc.tv_energy(g, f, delta) == pytest.approx(want, rel=1e-13)


@pytest.mark.parametrize("bc_xy,bc_z", BCS)
def test_P7_gradient_is_the_derivative_of_the_energy(orc, bc_xy, bc_z):
    """d = N_vox dE/df: central finite differences of the ENERGY routine, every voxel."""
    g = vol_geom(n=(5, 4, 4), bc_xy=bc_xy, bc_z=bc_z)
    rng = np.random.default_rng(1)
    f = rng.random(g.vol_shape)
    gg = rng.random(g.vol_shape)
    beta, delta = 3.7, 0.05
    d = orc.rof_gradient(g, f, gg, beta, delta)
    n = f.size
    eps = 1e-6
    for idx in np.ndindex(f.shape):
        fp = f.copy(); fp[idx] += eps
        fm = f.copy(); fm[idx] -= eps
        num = n * (orc.rof_energy(g, fp, gg, beta, delta) - orc.rof_energy(g, fm, gg, beta, delta)) / (2 * eps)
        assert d[idx] == pytest.approx(num, abs=2e-7 * max(1.0, abs(num))), idx


@pytest.mark.parametrize("bc_xy,bc_z", BCS)
def test_P7_divergence_is_negative_transpose_of_gradient(orc, bc_xy, bc_z):
    """<grad f, p> = -<f, div p> with p = grad q/|grad q|_delta: rof_gradient(gg=None) of q is -div p."""
    g = vol_geom(bc_xy=bc_xy, bc_z=bc_z)
    rng = np.random.default_rng(2)
    q = rng.random(g.vol_shape)
    f = rng.random(g.vol_shape)
    delta = 0.1
    qx, qy, qz = numpy_grad(q, g)
    nrm = np.sqrt(qx ** 2 + qy ** 2 + qz ** 2 + delta ** 2)
    fx, fy, fz = numpy_grad(f, g)
    lhs = (fx * qx / nrm + fy * qy / nrm + fz * qz / nrm).sum()
    minus_div = orc.rof_gradient(g, q, None, 0.0, delta)
    assert lhs == pytest.approx((f * minus_div).sum(), rel=1e-12)


def test_P8_tv_of_constants(orc):
    """(i) all-reflect: TV(c) = 0 exactly at delta = 0; (ii) paper BCs (zero in x,y, reflect in z):
    sum |grad f| = c [ (ny-1) nz / hx + (nx-1) nz / hy + nz sqrt(hx^-2 + hy^-2) ]."""
    c = 0.8
    g = vol_geom(bc_xy=I.BC_REFLECT, bc_z=I.BC_REFLECT)
    assert orc.tv_energy(g, np.full(g.vol_shape, c), 0.0) == 0.0
    g = vol_geom()
    nx, ny, nz = g.nx, g.ny, g.nz
    total = c * ((ny - 1) * nz / g.hx + (nx - 1) * nz / g.hy + nz * np.sqrt(g.hx ** -2 + g.hy ** -2))
    assert orc.tv_energy(g, np.full(g.vol_shape, c), 0.0) == pytest.approx(total / (nx * ny * nz), rel=1e-13)


def test_P9_every_accepted_step_satisfies_armijo(orc):
    """Re-run the prox one inner iteration at a time: the energy sequence strictly decreases and
    the report's first/last energies are those of g and of the returned f."""
    g = vol_geom(n=(12, 10, 8))
    rng = np.random.default_rng(3)
    gg = rng.random(g.vol_shape) * 0.03
    w = 2e-3
    fb = I.FbsSetup(eps_delta=1e-4, rel_tol=0.0, max_inner=1)
    energies = []
    for m in range(1, 7):
        f, rep = orc.tv_prox(g, gg, w, I.FbsSetup(eps_delta=1e-4, rel_tol=0.0, max_inner=m))
        assert rep.inner_iters == m
        assert rep.e_first == pytest.approx(orc.rof_energy(g, gg, gg, 1 / w, 1e-4), rel=1e-13)
        assert rep.e_last == pytest.approx(orc.rof_energy(g, f, gg, 1 / w, 1e-4), rel=1e-13)
        energies.append(rep.e_last)
    assert all(b < a for a, b in zip(energies, energies[1:]))
    assert energies[0] < rep.e_first
    # w = 0: identity
    f0, rep0 = orc.tv_prox(g, gg, 0.0, fb)
    assert np.array_equal(f0, gg) and rep0.inner_iters == 0


def test_P10_textbook_rof_two_plateaus_1d(orc):
    """1-D step, all-reflect, small delta: the exact ROF minimiser moves the plateaus of n_a and
    n_b voxels to a0 + w/(h n_a) and b0 - w/(h n_b).  Gradient descent is slow for small delta
    (step ~ delta), so delta = 1e-3 and 5000 inner steps: plateau means within 5 % of the shift,
    and the profile stays monotone with a sharp edge."""
    n_a, n_b, h = 12, 20, 1.5
    g = I.Geometry(nx=n_a + n_b, ny=1, nz=1, hx=h, hy=1.0, hz=1.0, nu=2, nv=2, du=1.0, dv=1.0,
                   n_proj=1, bc_xy=I.BC_REFLECT, bc_z=I.BC_REFLECT)
    a0, b0, w = 0.2, 1.0, 0.6
    gg = np.concatenate([np.full(n_a, a0), np.full(n_b, b0)]).reshape(g.vol_shape)
    f, rep = orc.tv_prox(g, gg, w, I.FbsSetup(eps_delta=1e-3, rel_tol=0.0, max_inner=5000,
                                              max_backtracks=60))
    f = f.ravel()
    sa, sb = w / (h * n_a), w / (h * n_b)
    assert abs(f[:n_a].mean() - (a0 + sa)) < 0.05 * sa
    assert abs(f[n_a:].mean() - (b0 - sb)) < 0.05 * sb
    assert np.all(np.diff(f) >= 0)      # the minimiser of a monotone step is monotone
    assert f[n_a] - f[n_a - 1] > 0.9 * (b0 - a0 - sa - sb) - 0.7 * (sa + sb)   # the edge survives


def test_P13_grid_transfers(orc):
    rng = np.random.default_rng(4)
    # restrict = 2x2x2 mean (numpy reshape definition); preserves the mean
    fine = rng.random((8, 6, 10))
    want = fine.reshape(4, 2, 3, 2, 5, 2).mean(axis=(1, 3, 5))
    np.testing.assert_allclose(orc.restrict(fine), want, rtol=0, atol=1e-15)
    # bin = 2x2 mean per view
    pr = rng.random((3, 6, 8))
    np.testing.assert_allclose(orc.bin2(pr), pr.reshape(3, 3, 2, 4, 2).mean(axis=(2, 4)), atol=1e-15)
    assert np.allclose(orc.bin2(np.full((2, 4, 4), 1.7)), 1.7)
    # prolong(const): const everywhere under reflect; const in the interior under zero BC in x,y
    c = np.full((4, 5, 6), 2.5)
    assert np.allclose(orc.prolong(c, I.BC_REFLECT, I.BC_REFLECT), 2.5)
    pz = orc.prolong(c, I.BC_ZERO, I.BC_REFLECT)
    assert np.allclose(pz[:, 1:-1, 1:-1], 2.5)
    assert np.allclose(pz[:, 0, 1:-1], 2.5 * 0.75) and np.allclose(pz[:, 0, 0], 2.5 * 0.75 ** 2)
    # linear ramps are reproduced in the interior (cell-centred coordinates), and
    # restrict(prolong(ramp)) == ramp in the interior
    z, y, x = np.meshgrid(np.arange(4), np.arange(5), np.arange(6), indexing="ij")
    ramp = 1.0 + 0.3 * x - 0.2 * y + 0.5 * z
    pf = orc.prolong(ramp, I.BC_REFLECT, I.BC_REFLECT)
    zf, yf, xf = np.meshgrid(np.arange(8), np.arange(10), np.arange(12), indexing="ij")
    want = 1.0 + 0.3 * ((xf + 0.5) / 2 - 0.5) - 0.2 * ((yf + 0.5) / 2 - 0.5) + 0.5 * ((zf + 0.5) / 2 - 0.5)
    np.testing.assert_allclose(pf[1:-1, 1:-1, 1:-1], want[1:-1, 1:-1, 1:-1], atol=1e-14)
    np.testing.assert_allclose(orc.restrict(pf)[1:-1, 1:-1, 1:-1], ramp[1:-1, 1:-1, 1:-1], atol=1e-14)
    # prolongation preserves the mean of interior-supported volumes (zero BC)
    blob = np.zeros((4, 6, 6)); blob[1:3, 2:4, 2:4] = rng.random((2, 2, 2))
    assert orc.prolong(blob, I.BC_ZERO, I.BC_ZERO).mean() == pytest.approx(blob.mean(), rel=1e-13)


def _replay_prox(orc, g, gg, w, c, alpha, eps, max_inner, delta, max_bt=20):
    """The loop of PAPER.md:L155-L159 spelled out once more on top of the two pinned primitives (rof_energy: P8 and
    the numpy definition; rof_gradient: P7 finite differences): start at f = g, first trial step 1/beta, Eq. 5
    `E_new <= E0 - c lam mean(d^2)` else lam <- alpha lam, stop when |E_new - E0| / E0 < eps.  Returns the counts, the
    relative distance of every trial from the Armijo threshold and the relative decrease of every accepted step."""
    beta = 1.0 / w
    f = gg.copy()
    e0 = orc.rof_energy(g, f, gg, beta, delta)
    inner = trials = 0
    margins, rels = [], []
    for _ in range(max_inner):
        d = orc.rof_gradient(g, f, gg, beta, delta)
        dm = float(np.mean(d * d))
        lam, ok = w, False
        for _bt in range(max_bt + 1):
            en = orc.rof_energy(g, f - lam * d, gg, beta, delta)
            trials += 1
            margins.append((en - (e0 - c * lam * dm)) / e0)
            if en <= e0 - c * lam * dm:
                ok = True
                break
            lam *= alpha
        if not ok:
            break
        f = f - lam * d
        inner += 1
        rels.append(abs(en - e0) / e0)
        e0 = en
        if rels[-1] < eps:
            break
    return inner, trials, margins, rels, f


@pytest.mark.parametrize("w,c,alpha", [(2e-3, 0.01, 0.6), (2e-2, 0.01, 0.6), (2e-2, 0.5, 0.6), (0.2, 0.9, 0.6), (2e-2, 0.5, 0.3)])
def test_P9b_armijo_constant_and_shrink_decide_the_trial_count(orc, w, c, alpha):
    """Eq. 5 with its constant c and the shrink factor alpha (L159): the first trial step 1/beta
    overshoots, so the accepted step is reached after a KNOWN number of rejected trials, each of which misses the
    threshold E0 - c lam mean(d^2) by a margin far from a tie.  An oracle that dropped c (accepted any decrease), put it
    on the wrong term or shrank by another factor returns other counts."""
    g = vol_geom(n=(12, 10, 8))
    gg = np.random.default_rng(3).random(g.vol_shape) * 0.03
    inner, trials, margins, _, f_want = _replay_prox(orc, g, gg, w, c, alpha, 0.0, 3, 1e-4)
    assert inner == 3 and trials > inner                       # backtracking happened
    assert min(abs(m) for m in margins) > 5e-5                 # no trial sits on the threshold
    f, rep = orc.tv_prox(g, gg, w, I.FbsSetup(eps_delta=1e-4, rel_tol=0.0, max_inner=3, armijo_c=c, shrink_alpha=alpha))
    assert (rep.inner_iters, rep.trials) == (inner, trials)
    np.testing.assert_allclose(f, f_want, rtol=0, atol=1e-15)


def test_P9b_the_constant_matters(orc):
    """Same problem, c = 0.01 (L159) against c = 0.9: some trials decrease the energy but not by c lam mean(d^2)."""
    g = vol_geom(n=(12, 10, 8))
    gg = np.random.default_rng(3).random(g.vol_shape) * 0.03
    t = {}
    for c in (0.0, 0.01, 0.9):
        _, rep = orc.tv_prox(g, gg, 2e-3, I.FbsSetup(eps_delta=1e-4, rel_tol=0.0, max_inner=3, armijo_c=c))
        t[c] = rep.trials
    assert t[0.0] <= t[0.01] < t[0.9]
    assert (t[0.01], t[0.9]) == (5, 15)


def test_P9c_epsilon_stop_uses_the_relative_decrease_of_the_step(orc):
    """The stop |E_new - E0| / E0 < eps (eps = 1e-3 there): eps placed between the relative decreases
    of two known accepted steps stops exactly there; and the denominator is the energy BEFORE the step -- an eps between
    |dE|/E0 and |dE|/E_new tells the two apart."""
    g = vol_geom(n=(12, 10, 8))
    gg = np.random.default_rng(3).random(g.vol_shape) * 0.03
    w = 2e-2
    _, _, _, rels, _ = _replay_prox(orc, g, gg, w, 0.01, 0.6, 0.0, 12, 1e-4)
    assert rels[1] < 0.07 < rels[0] and min(rels[:5]) > 0.05 > rels[5]      # the fixture this test is built on
    for eps, want in ((0.07, 2), (0.05, 6)):
        inner, trials, _, _, f_want = _replay_prox(orc, g, gg, w, 0.01, 0.6, eps, 50, 1e-4)
        assert inner == want
        f, rep = orc.tv_prox(g, gg, w, I.FbsSetup(eps_delta=1e-4, rel_tol=eps, max_inner=50))
        assert (rep.inner_iters, rep.trials) == (inner, trials)
        np.testing.assert_allclose(f, f_want, rtol=0, atol=1e-15)
    # between |dE|/E0 = rels[1] and |dE|/E_new = rels[1] / (1 - rels[1]): stops at step 2 only with E0 below the line
    eps = 0.5 * (rels[1] + rels[1] / (1.0 - rels[1]))
    _, rep = orc.tv_prox(g, gg, w, I.FbsSetup(eps_delta=1e-4, rel_tol=eps, max_inner=50))
    assert rep.inner_iters == 2
    _, rep = orc.tv_prox(g, gg, w, I.FbsSetup(eps_delta=1e-4, rel_tol=0.999 * rels[1], max_inner=50))
    assert rep.inner_iters > 2
