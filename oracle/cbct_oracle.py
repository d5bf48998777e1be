"""ctypes front-end of the CPU oracle `cbct_oracle.c` (numpy in, numpy out, float64).

TEST INFRASTRUCTURE ONLY: tests/, `__graft_entry__.smoke()` and the `cpu_baseline` /
`--impl reference` legs of `bench.py` may import this.  The product path
(`paper_1001_0599_b200`) never does, and this module never imports the product's
kernels or binding -- it takes the plain `Geometry` description objects of
`paper_1001_0599_b200.inputs` by duck typing only (attribute access).

Every function cites the passage of PAPER.md that the C routine follows; the
arithmetic lives in the C file, this file only marshals arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cbct_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_cbct.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (+OpenMP).  Returns the library path."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


class _OGeom(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("hx", C.c_double), ("hy", C.c_double), ("hz", C.c_double),
                ("off", C.c_double * 3),
                ("nu", C.c_int), ("nv", C.c_int),
                ("du", C.c_double), ("dv", C.c_double), ("offu", C.c_double), ("offv", C.c_double),
                ("sad", C.c_double), ("sdd", C.c_double),
                ("n_proj", C.c_int), ("angles", C.POINTER(C.c_double)),
                ("bc_xy", C.c_int), ("bc_z", C.c_int)]


class _TvParams(C.Structure):
    _fields_ = [("eps_delta", C.c_double), ("max_inner", C.c_int), ("max_backtracks", C.c_int),
                ("armijo_c", C.c_double), ("shrink_alpha", C.c_double), ("rel_tol", C.c_double)]


class _TvReport(C.Structure):
    _fields_ = [("inner_iters", C.c_int), ("trials", C.c_int),
                ("e_first", C.c_double), ("e_last", C.c_double)]


@dataclass
class TvReport:
    inner_iters: int
    trials: int
    e_first: float
    e_last: float


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_ray_box_len.restype = C.c_double
        _lib.oracle_forward.restype = C.c_long
        _lib.oracle_tv_energy.restype = C.c_double
        _lib.oracle_rof_energy.restype = C.c_double
        _lib.oracle_step_bound.restype = C.c_double
        _lib.oracle_fbs_level.restype = C.c_double
        _lib.oracle_threads.restype = C.c_int
    return _lib


def threads() -> int:
    return int(lib().oracle_threads())


def _arr(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _p(a):
    return a.ctypes.data_as(_dp)


def _geom(g):
    """Geometry description -> (C struct, keep-alive)."""
    ang = np.ascontiguousarray(g.angles_rad(), dtype=np.float64)
    s = _OGeom()
    s.nx, s.ny, s.nz = g.nx, g.ny, g.nz
    s.hx, s.hy, s.hz = g.hx, g.hy, g.hz
    s.off[0], s.off[1], s.off[2] = (float(x) for x in g.vol_off)
    s.nu, s.nv, s.du, s.dv = g.nu, g.nv, g.du, g.dv
    s.offu, s.offv = g.det_off_u, g.det_off_v
    s.sad, s.sdd, s.n_proj = g.sad, g.sdd, g.n_proj
    s.angles = _p(ang)
    s.bc_xy, s.bc_z = g.bc_xy, g.bc_z
    return s, ang


def _tvp(fbs):
    return _TvParams(fbs.eps_delta, fbs.max_inner, fbs.max_backtracks, fbs.armijo_c,
                     fbs.shrink_alpha, fbs.rel_tol)


# -- geometry ---------------------------------------------------------------

def ray(g, a, iu, iv):
    """Source S and vector D = P(u,v) - S (Eq. 1, L374 Eq. A2)."""
    s, keep = _geom(g)
    S = np.zeros(3); D = np.zeros(3)
    lib().oracle_ray(C.byref(s), int(a), int(iu), int(iv), _p(S), _p(D))
    return S, D


def voxel_to_detector(g, a, X):
    """(u*, v*, l) of Eq. A6 for a general view."""
    s, keep = _geom(g)
    X = _arr(X, (3,))
    u = C.c_double(); v = C.c_double(); l = C.c_double()
    lib().oracle_voxel_to_detector(C.byref(s), int(a), _p(X), C.byref(u), C.byref(v), C.byref(l))
    return u.value, v.value, l.value


def ray_box_len(S, D, lo, hi) -> float:
    S, D, lo, hi = (_arr(x, (3,)) for x in (S, D, lo, hi))
    return float(lib().oracle_ray_box_len(_p(S), _p(D), _p(lo), _p(hi)))


# -- projectors -------------------------------------------------------------

def forward_brute(g, f):
    """P f by definition: every voxel's ray/box length (Eq. 1; L187)."""
    s, keep = _geom(g)
    f = _arr(f, g.vol_shape)
    p = np.zeros(g.proj_shape)
    lib().oracle_forward_brute(C.byref(s), _p(f), _p(p))
    return p


def back_brute(g, p):
    """P^T p by definition (gather over every ray)."""
    s, keep = _geom(g)
    p = _arr(p, g.proj_shape)
    b = np.zeros(g.vol_shape)
    lib().oracle_back_brute(C.byref(s), _p(p), _p(b))
    return b


def forward(g, f, return_samples=False):
    """P f by incremental (Siddon) traversal, L187/L243.  Optionally also S."""
    s, keep = _geom(g)
    f = _arr(f, g.vol_shape)
    p = np.zeros(g.proj_shape)
    n = lib().oracle_forward(C.byref(s), _p(f), _p(p))
    return (p, int(n)) if return_samples else p


def back(g, p):
    """Exact transpose of `forward` (scatter along each ray, L187-L191)."""
    s, keep = _geom(g)
    p = _arr(p, g.proj_shape)
    b = np.zeros(g.vol_shape)
    lib().oracle_back(C.byref(s), _p(p), _p(b))
    return b


def back_eq6(g, T):
    """The paper's closed-form gradient Eq. 6 (L195-L199): voxel-driven, bilinear T, on the scale of P^T T."""
    s, keep = _geom(g)
    T = _arr(T, g.proj_shape)
    b = np.zeros(g.vol_shape)
    lib().oracle_back_eq6(C.byref(s), _p(T), _p(b))
    return b


# -- TV / ROF ---------------------------------------------------------------

def tv_energy(g, f, delta) -> float:
    """E1^delta = mean |grad f|_delta (L100, reading S6)."""
    s, keep = _geom(g)
    f = _arr(f, g.vol_shape)
    return float(lib().oracle_tv_energy(C.byref(s), _p(f), C.c_double(delta)))


def rof_energy(g, f, gg, beta, delta) -> float:
    """E_ROF = E1 + (beta/2) E3 (L151, L155)."""
    s, keep = _geom(g)
    f = _arr(f, g.vol_shape); gg = _arr(gg, g.vol_shape)
    return float(lib().oracle_rof_energy(C.byref(s), _p(f), _p(gg), C.c_double(beta),
                                         C.c_double(delta)))


def rof_gradient(g, f, gg, beta, delta):
    """d = N_vox dE_ROF/df = -div p + beta (f - g) (L155); gg=None => TV part only."""
    s, keep = _geom(g)
    f = _arr(f, g.vol_shape)
    d = np.zeros(g.vol_shape)
    if gg is None:
        lib().oracle_rof_gradient(C.byref(s), _p(f), None, C.c_double(0.0), C.c_double(delta), _p(d))
    else:
        gg = _arr(gg, g.vol_shape)
        lib().oracle_rof_gradient(C.byref(s), _p(f), _p(gg), C.c_double(beta), C.c_double(delta),
                                  _p(d))
    return d


def tv_prox(g, gg, w, fbs):
    """TV-prox_w(g) by Armijo gradient descent (L155-L159).  Returns (f, TvReport)."""
    s, keep = _geom(g)
    gg = _arr(gg, g.vol_shape)
    f = np.zeros(g.vol_shape)
    tp = _tvp(fbs)
    rep = _TvReport()
    lib().oracle_tv_prox(C.byref(s), _p(gg), _p(f), C.c_double(w), C.byref(tp), C.byref(rep))
    return f, TvReport(rep.inner_iters, rep.trials, rep.e_first, rep.e_last)


# -- transfers --------------------------------------------------------------

def restrict(fine):
    fine = _arr(fine)
    nz, ny, nx = fine.shape
    out = np.zeros((nz // 2, ny // 2, nx // 2))
    lib().oracle_restrict(nx, ny, nz, _p(fine), _p(out))
    return out


def bin2(proj):
    proj = _arr(proj)
    n_p, nv, nu = proj.shape
    out = np.zeros((n_p, nv // 2, nu // 2))
    lib().oracle_bin(nu, nv, n_p, _p(proj), _p(out))
    return out


def prolong(coarse, bc_xy, bc_z):
    coarse = _arr(coarse)
    cz, cy, cx = coarse.shape
    out = np.zeros((2 * cz, 2 * cy, 2 * cx))
    lib().oracle_prolong(cx, cy, cz, int(bc_xy), int(bc_z), _p(coarse), _p(out))
    return out


# -- quality metrics (NEXT-3) -------------------------------------------------

def quality_metrics(f, f0):
    """The paper's metrics (L263) written out: e = ||f - f0||_2 / ||f0||_2 and the Pearson correlation
    c = sum (f - mean f)(f0 - mean f0) / sqrt(sum (f - mean f)^2 sum (f0 - mean f0)^2), in fp64."""
    f = np.asarray(f, dtype=np.float64).ravel()
    f0 = np.asarray(f0, dtype=np.float64).ravel()
    e = float(np.sqrt(np.sum((f - f0) ** 2) / np.sum(f0 ** 2)))
    a, b = f - f.mean(), f0 - f0.mean()
    c = float(np.sum(a * b) / np.sqrt(np.sum(a * a) * np.sum(b * b)))
    return e, c


# -- FBS --------------------------------------------------------------------

def step_bound(g) -> float:
    """Lhat = c_norm max_v [P^T P 1]_v (reading S5)."""
    s, keep = _geom(g)
    return float(lib().oracle_step_bound(C.byref(s)))


@dataclass
class FbsResult:
    f: np.ndarray
    objective: np.ndarray
    step_abs: np.ndarray
    inner_total: int
    trials_total: int
    iters_done: tuple = ()


def fbs(g, y, fbs_setup, f0=None):
    """Algorithm A1 with the multi-grid driver (L137-L151, L215-L223)."""
    s, keep = _geom(g)
    y = _arr(y, g.proj_shape)
    iters = np.ascontiguousarray(fbs_setup.iters_per_level, dtype=np.int32)
    n_levels = len(iters)
    f = np.zeros(g.vol_shape) if f0 is None else _arr(f0, g.vol_shape).copy()
    obj = np.zeros(int(iters.sum()))
    step_abs = np.zeros(n_levels)
    tp = _tvp(fbs_setup)
    inner = C.c_int(0); trials = C.c_int(0)
    done = np.zeros(n_levels, dtype=np.int32)
    lib().oracle_fbs(C.byref(s), _p(y), _p(f), C.c_double(fbs_setup.tv_weight),
                     C.c_double(fbs_setup.step), n_levels, iters.ctypes.data_as(C.POINTER(C.c_int)),
                     int(bool(fbs_setup.nonneg)), int(f0 is not None),
                     int(getattr(fbs_setup, "backprojector", 0)),
                     C.c_double(float(getattr(fbs_setup, "conv_tol", 0.0))), C.byref(tp), _p(obj),
                     _p(step_abs), C.byref(inner), C.byref(trials), done.ctypes.data_as(C.POINTER(C.c_int)))
    return FbsResult(f, obj[:int(done.sum())], step_abs, inner.value, trials.value, tuple(int(x) for x in done))
