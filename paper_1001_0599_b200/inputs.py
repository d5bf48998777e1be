"""Seeded synthetic inputs for the cone-beam CT hot path (numpy only).

This module is the ONE piece shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_1001_0599_b200/csrc`): it builds problem descriptions and input
arrays -- geometry descriptors, ellipsoid phantoms, simulated projection data,
Poisson noise -- and holds none of the method's arithmetic (no projector over a
voxel grid, no TV, no FBS, no grid transfer).  It imports neither side.

Conventions (Eq. 1, L374 A2):
  * world z = rotation axis; view angle theta: e_n=(cos,sin,0), e_u=(sin,-cos,0),
    e_v=(0,0,1); source S=-SAD*e_n; detector point P(u,v)=S+SDD*e_n+u*e_u+v*e_v.
  * volume index (k*ny+j)*nx+i, voxel centre x_i=(i-(nx-1)/2)*hx+off_x.
  * projections index (p*nv+jv)*nu+iu, pixel centre u_i=(i-(nu-1)/2)*du+off_u.

The paper measures on the NCAT phantom, a CatPhan 600, a patient scan and a
Rando phantom.  None of them is available;
the seeded ellipsoid phantoms below take their sizes (256^3-class volumes,
512x384 imager, SAD 1000 / SDD 1500 mm, 40-360 views over 360 degrees,
attenuation 0-0.05 /mm, low-count Poisson noise) and stand in for them.
The 10-ellipsoid head-like table for config 1 is this repository's own.
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

BC_ZERO = 0
BC_REFLECT = 1

SEED_BASE = 10010599  # phantom seed = SEED_BASE + k for config k; noise seed = +100


@dataclass
class Geometry:
    """Plain description of one circular cone-beam acquisition (all lengths in mm)."""
    nx: int
    ny: int
    nz: int
    hx: float
    hy: float
    hz: float
    nu: int
    nv: int
    du: float
    dv: float
    sad: float = 1000.0
    sdd: float = 1500.0
    n_proj: int = 1
    vol_off: Sequence[float] = (0.0, 0.0, 0.0)
    det_off_u: float = 0.0
    det_off_v: float = 0.0
    angles: Optional[np.ndarray] = None  # radians; None => 2*pi*k/n_proj
    bc_xy: int = BC_ZERO      # PAPER.md:L161 zero BC along AP / lateral
    bc_z: int = BC_REFLECT    # PAPER.md:L161 reflective BC along SI

    def angles_rad(self) -> np.ndarray:
        if self.angles is not None:
            a = np.ascontiguousarray(self.angles, dtype=np.float64)
            assert a.shape == (self.n_proj,)
            return a
        return 2.0 * np.pi * np.arange(self.n_proj, dtype=np.float64) / self.n_proj

    @property
    def vol_shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def proj_shape(self):
        return (self.n_proj, self.nv, self.nu)

    def replace(self, **kw) -> "Geometry":
        return dataclasses.replace(self, **kw)


@dataclass
class Ellipsoid:
    """Additive ellipsoid: adds `value` (1/mm) inside; rotated by `phi` about z."""
    centre: Sequence[float]
    axes: Sequence[float]
    phi: float
    value: float


@dataclass
class FbsSetup:
    """Iteration parameters of one config."""
    tv_weight: float = 0.01
    step: float = 1.0
    iters_per_level: Sequence[int] = (20,)
    nonneg: bool = True
    eps_delta: float = 1e-5
    max_inner: int = 20
    max_backtracks: int = 20
    armijo_c: float = 0.01
    shrink_alpha: float = 0.6
    rel_tol: float = 1e-3
    backprojector: int = 0    # 0: exact transpose P^T (matched pair); 1: the paper's Eq. 6
    conv_tol: float = 0.0     # > 0: a level stops once ||f_new - f_old|| <= conv_tol ||f_old||


@dataclass
class Config:
    name: str
    geom: Geometry
    fbs: FbsSetup
    ellipsoids: list = field(default_factory=list)
    photons: Optional[float] = None   # incident photons per pixel; None => noiseless
    seed: int = SEED_BASE


# --------------------------------------------------------------------------
# phantoms
# --------------------------------------------------------------------------

def headlike_phantom(half: float = 32.0) -> list:
    """This repository's own 10-ellipsoid head-like table (config 1).

    Lengths are fractions of `half` (half the cube edge, mm).  Values are signed
    increments; every point's total lies in [0, 0.02] /mm.
    """
    t = [
        # centre (x,y,z)          semi-axes            phi(deg) increment
        ((0.00, 0.00, 0.00), (0.70, 0.88, 0.84), 0.0, 0.0200),   # bone-like shell
        ((0.00, -0.02, 0.00), (0.64, 0.82, 0.78), 0.0, -0.0100),  # interior -> 0.010
        ((0.24, 0.04, -0.05), (0.12, 0.34, 0.30), 15.0, -0.0040),  # lateral lobe
        ((-0.24, 0.04, -0.05), (0.16, 0.40, 0.32), -15.0, -0.0040),  # lateral lobe
        ((0.00, 0.36, 0.10), (0.22, 0.26, 0.30), 0.0, 0.0030),   # upper mass
        ((0.00, 0.08, 0.20), (0.10, 0.10, 0.14), 0.0, 0.0040),   # central sphere-ish
        ((0.00, -0.14, -0.20), (0.09, 0.09, 0.12), 0.0, 0.0040),
        ((-0.14, -0.58, 0.00), (0.10, 0.06, 0.12), 30.0, 0.0050),  # small inclusions
        ((0.02, -0.60, 0.25), (0.07, 0.07, 0.07), 0.0, 0.0050),
        ((0.16, -0.56, -0.30), (0.06, 0.10, 0.09), -40.0, 0.0050),
    ]
    return [Ellipsoid(tuple(half * c for c in ce), tuple(half * a for a in ax),
                      np.deg2rad(ph), val) for ce, ax, ph, val in t]


def random_ellipsoids(rng: np.random.Generator, n: int, half_extent: Sequence[float],
                      axes_range=(5.0, 40.0), value_range=(0.0, 0.010),
                      inner_frac: float = 0.8) -> list:
    """n additive ellipsoids; draw order per ellipsoid: centre xyz, axes xyz, phi, value."""
    out = []
    hx, hy, hz = half_extent
    for _ in range(n):
        c = rng.uniform(-inner_frac, inner_frac, size=3) * np.array([hx, hy, hz])
        a = rng.uniform(axes_range[0], axes_range[1], size=3)
        phi = rng.uniform(0.0, np.pi)
        val = rng.uniform(value_range[0], value_range[1])
        out.append(Ellipsoid(tuple(c), tuple(a), float(phi), float(val)))
    return out


def paint(ellipsoids, geom: Geometry) -> np.ndarray:
    """Sample the additive phantom at voxel centres -> float32 [nz,ny,nx]."""
    x = (np.arange(geom.nx) - (geom.nx - 1) / 2.0) * geom.hx + geom.vol_off[0]
    y = (np.arange(geom.ny) - (geom.ny - 1) / 2.0) * geom.hy + geom.vol_off[1]
    z = (np.arange(geom.nz) - (geom.nz - 1) / 2.0) * geom.hz + geom.vol_off[2]
    vol = np.zeros(geom.vol_shape, dtype=np.float64)
    for e in ellipsoids:
        cx, cy, cz = e.centre
        ax, ay, az = e.axes
        # bounding box in index space keeps this cheap on big grids
        r = max(ax, ay)
        ix = np.where(np.abs(x - cx) <= r)[0]
        iy = np.where(np.abs(y - cy) <= r)[0]
        iz = np.where(np.abs(z - cz) <= az)[0]
        if len(ix) == 0 or len(iy) == 0 or len(iz) == 0:
            continue
        X = x[ix][None, None, :] - cx
        Y = y[iy][None, :, None] - cy
        Z = z[iz][:, None, None] - cz
        c, s = np.cos(e.phi), np.sin(e.phi)
        xr = (c * X + s * Y) / ax
        yr = (-s * X + c * Y) / ay
        zr = Z / az
        inside = (xr * xr + yr * yr + zr * zr) <= 1.0
        vol[np.ix_(iz, iy, ix)] += e.value * inside
    return vol.astype(np.float32)


def analytic_projections(ellipsoids, geom: Geometry) -> np.ndarray:
    """Closed-form line integrals of the additive ellipsoid phantom -> float64 [p,nv,nu].

    Ray for pixel (iu,iv) of view p runs from the source to the pixel centre
    (Eq. 1).  For one ellipsoid, map to its unit sphere: with
    S' and D' the transformed source and direction, A=|D'|^2, B=S'.D',
    C=|S'|^2-1, the chord is L*2*sqrt(B^2-A*C)/A when the discriminant is positive.
    """
    ang = geom.angles_rad()
    u = (np.arange(geom.nu) - (geom.nu - 1) / 2.0) * geom.du + geom.det_off_u
    v = (np.arange(geom.nv) - (geom.nv - 1) / 2.0) * geom.dv + geom.det_off_v
    U, V = np.meshgrid(u, v)  # [nv,nu]
    out = np.zeros(geom.proj_shape, dtype=np.float64)
    for p, th in enumerate(ang):
        c, s = np.cos(th), np.sin(th)
        S = np.array([-geom.sad * c, -geom.sad * s, 0.0])
        Dx = geom.sdd * c + U * s
        Dy = geom.sdd * s - U * c
        Dz = V
        L = np.sqrt(Dx * Dx + Dy * Dy + Dz * Dz)
        acc = np.zeros_like(U)
        for e in ellipsoids:
            ce, se = np.cos(e.phi), np.sin(e.phi)
            ax, ay, az = e.axes
            sx, sy, sz = S - np.asarray(e.centre, dtype=np.float64)
            spx = (ce * sx + se * sy) / ax
            spy = (-se * sx + ce * sy) / ay
            spz = sz / az
            dpx = (ce * Dx + se * Dy) / ax
            dpy = (-se * Dx + ce * Dy) / ay
            dpz = Dz / az
            A = dpx * dpx + dpy * dpy + dpz * dpz
            B = spx * dpx + spy * dpy + spz * dpz
            C = spx * spx + spy * spy + spz * spz - 1.0
            disc = B * B - A * C
            chord = np.where(disc > 0.0, 2.0 * np.sqrt(np.maximum(disc, 0.0)) / A, 0.0)
            acc += e.value * L * chord
        out[p] = acc
    return out


def poisson_log(p: np.ndarray, photons: float, seed: int) -> np.ndarray:
    """y = ln(I0 / max(N,1)),  N ~ Poisson(I0 * exp(-p))."""
    rng = np.random.default_rng(seed)
    lam = photons * np.exp(-np.asarray(p, dtype=np.float64))
    n = rng.poisson(lam).astype(np.float64)
    return np.log(photons / np.maximum(n, 1.0))


def uniform_volume(geom: Geometry, seed: int, hi: float = 0.03) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return (rng.random(geom.vol_shape, dtype=np.float32) * np.float32(hi)).astype(np.float32)


def uniform_projections(geom: Geometry, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return rng.random(geom.proj_shape, dtype=np.float32)


# --------------------------------------------------------------------------
# the five configs of BASELINE.json
# --------------------------------------------------------------------------

def _cone(n, h, nu, nv, pitch, n_proj, nz=None, hz=None) -> Geometry:
    return Geometry(nx=n, ny=n, nz=n if nz is None else nz, hx=h, hy=h,
                    hz=h if hz is None else hz, nu=nu, nv=nv, du=pitch, dv=pitch,
                    sad=1000.0, sdd=1500.0, n_proj=n_proj)


def config(k: int) -> Config:
    """Config k=1..4 of BASELINE.json (config 5 is the sweep: see `sweep_geometry`)."""
    seed = SEED_BASE + k
    rng = np.random.default_rng(seed)
    if k == 1:
        g = _cone(32, 2.0, 48, 48, 1.6, 8)
        return Config("tiny-headlike-32", g, FbsSetup(iters_per_level=(20,)),
                      headlike_phantom(32.0), None, seed)
    if k == 2:
        g = _cone(128, 2.0, 256, 192, 1.55, 40)
        ell = [Ellipsoid((0.0, 0.0, 0.0), (112.0, 92.0, 122.0), 0.0, 0.02)]
        ell += random_ellipsoids(rng, 30, (128.0, 128.0, 128.0))
        return Config("random-ellipsoids-128", g, FbsSetup(iters_per_level=(50, 50)),
                      ell, 1e5, seed)
    if k == 3:
        g = _cone(256, 1.0, 512, 384, 0.776, 40)
        ell = [
            Ellipsoid((0.0, 0.0, 0.0), (118.0, 88.0, 125.0), 0.0, 0.02),       # body
            Ellipsoid((52.0, 6.0, 10.0), (38.0, 52.0, 80.0), 0.0, -0.018),     # lung -> 0.002
            Ellipsoid((-52.0, 6.0, 10.0), (38.0, 52.0, 80.0), 0.0, -0.018),    # lung -> 0.002
            Ellipsoid((0.0, -58.0, 0.0), (14.0, 14.0, 124.0), 0.0, 0.02),      # spine -> 0.04
        ]
        ell += random_ellipsoids(rng, 40, (128.0, 128.0, 128.0), axes_range=(4.0, 30.0),
                                 value_range=(0.0, 0.008), inner_frac=0.6)
        return Config("torso-256", g, FbsSetup(iters_per_level=(100, 100, 100)),
                      ell, 5e4, seed)
    if k == 4:
        g = _cone(512, 0.5, 512, 384, 0.776, 360, nz=256, hz=1.0)
        ell = [
            Ellipsoid((0.0, 0.0, 0.0), (92.0, 112.0, 120.0), 0.0, 0.05),       # skull
            Ellipsoid((0.0, 0.0, 0.0), (85.0, 105.0, 113.0), 0.0, -0.03),      # brain -> 0.02
        ]
        ell += random_ellipsoids(rng, 60, (128.0, 128.0, 128.0), axes_range=(3.0, 25.0),
                                 value_range=(-0.004, 0.006), inner_frac=0.45)
        return Config("head-512x512x256", g, FbsSetup(iters_per_level=(100, 100, 100)),
                      ell, 5e3, seed)
    raise ValueError("config k must be 1..4 (config 5 is the sweep)")


def sweep_geometry(n: int, n_proj: int) -> Geometry:
    """Config 5: n^3 volume with a fixed 256 mm field of view, 512x384 imager."""
    return _cone(n, 256.0 / n, 512, 384, 0.776, n_proj)


def make_projections(cfg: Config) -> np.ndarray:
    """Projection data y of a config -> float32 [p,nv,nu] (analytic integrals + noise)."""
    p = analytic_projections(cfg.ellipsoids, cfg.geom)
    if cfg.photons is not None:
        p = poisson_log(p, cfg.photons, cfg.seed + 100)
    return np.ascontiguousarray(p, dtype=np.float32)
