"""NEXT-3: the paper's image-quality metrics e and c.  The oracle writes the definitions out;
it is pinned by values worked by hand, closed forms and numpy's library routine; the CUDA reduction is compared
with it on seeded volumes."""
import numpy as np
import pytest

from paper_1001_0599_b200 import inputs as I


def test_oracle_metrics_hand_values_and_closed_forms(orc):
    f0 = np.array([1.0, 2.0, 3.0, 4.0])
    f = np.array([1.0, 2.0, 3.0, 6.0])
    e, c = orc.quality_metrics(f, f0)
    assert e == pytest.approx(2.0 / np.sqrt(30.0), rel=1e-14)          # ||(0,0,0,2)|| / ||(1,2,3,4)||
    # by hand: means 3 and 2.5; sum (f-3)(f0-2.5) = 3+0.5+0+4.5 = 8; sum (f-3)^2 = 14; sum (f0-2.5)^2 = 5
    assert c == pytest.approx(8.0 / np.sqrt(14.0 * 5.0), rel=1e-14)
    rng = np.random.default_rng(5)
    g0 = rng.random(1000)
    # an affine image of the truth is perfectly (anti-)correlated; e follows in closed form
    for a, b in [(2.0, 0.3), (-0.5, 1.0)]:
        e, c = orc.quality_metrics(a * g0 + b, g0)
        assert c == pytest.approx(np.sign(a), abs=1e-12)
        assert e == pytest.approx(np.linalg.norm((a - 1) * g0 + b) / np.linalg.norm(g0), rel=1e-12)
    g1 = rng.random(1000)
    e, c = orc.quality_metrics(g1, g0)
    assert c == pytest.approx(np.corrcoef(g1, g0)[0, 1], rel=1e-12)     # the library's Pearson coefficient
    assert orc.quality_metrics(g0, g0) == (0.0, pytest.approx(1.0, abs=1e-15))


@pytest.mark.gpu
@pytest.mark.parametrize("shape", [(19, 45, 37), (64, 64, 64)])
def test_gpu_metrics_match_oracle(orc, shape):
    import torch
    from paper_1001_0599_b200 import cbct
    nz, ny, nx = shape
    g = I.Geometry(nx=nx, ny=ny, nz=nz, hx=1.0, hy=1.0, hz=1.0, nu=16, nv=16, du=4.0, dv=4.0, n_proj=2)
    f0 = I.uniform_volume(g, 81)
    f = (f0 * 0.9 + 0.002 * I.uniform_volume(g, 82, hi=1.0)).astype(np.float32)
    we, wc = orc.quality_metrics(f, f0)
    with cbct.geometry_create(g) as h:
        a, b = torch.from_numpy(f).cuda(), torch.from_numpy(f0).cuda()
        e, c = h.quality_metrics(a, b)
        e2, c2 = h.quality_metrics(a, b)
        assert h.quality_metrics(b, b) == (0.0, pytest.approx(1.0, abs=1e-12))
    assert e == pytest.approx(we, rel=1e-10) and c == pytest.approx(wc, rel=1e-10)
    assert (e, c) == (e2, c2)                                             # fixed summation order
