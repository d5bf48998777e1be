"""Thin ctypes binding of libcbct (include/cbct.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch is used for device
memory and streams.  There is no CPU fallback: importing works anywhere (so that the
exported symbols can be checked without a GPU), but creating a `Geometry` handle fails
loudly when the library or an sm_100 device is missing.

Function names mirror the C ABI: geometry_create / forward_project / back_project /
tv_prox / fbs_reconstruct (+ the grid transfers, step_bound, tv_energy).
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))

CBCT_OK = 0
STATUS_NAMES = {0: "CBCT_OK", 1: "CBCT_ERR_INVALID_ARG", 2: "CBCT_ERR_GEOMETRY", 3: "CBCT_ERR_CUDA",
                4: "CBCT_ERR_OOM", 5: "CBCT_ERR_UNSUPPORTED"}

# every symbol include/cbct.h declares
EXPORTS = [
    "cbct_geometry_create", "cbct_geometry_destroy", "cbct_geometry_symmetry", "cbct_geometry_device_bytes",
    "cbct_geometry_back_path", "cbct_bound_violations",
    "cbct_forward_project", "cbct_back_project", "cbct_back_project_eq6", "cbct_count_samples", "cbct_step_bound", "cbct_tv_prox", "cbct_tv_energy",
    "cbct_quality_metrics", "cbct_quality_metrics_static",
    "cbct_restrict_volume", "cbct_bin_projections", "cbct_prolong_volume",
    "cbct_fbs_reconstruct", "cbct_fbs_reconstruct_host", "cbct_fbs_reconstruct_sharded", "cbct_shard_range",
    "cbct_shard_units", "cbct_launch_count",
    "cbct_set_stage_timing", "cbct_get_stage_ms", "cbct_gather_ceiling", "cbct_last_error", "cbct_version",
]


class CbctError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


class _Desc(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("hx", C.c_double), ("hy", C.c_double), ("hz", C.c_double),
                ("vol_off", C.c_double * 3),
                ("nu", C.c_int), ("nv", C.c_int),
                ("du", C.c_double), ("dv", C.c_double), ("det_off_u", C.c_double), ("det_off_v", C.c_double),
                ("sad", C.c_double), ("sdd", C.c_double),
                ("n_proj", C.c_int), ("angles_rad", C.POINTER(C.c_double)),
                ("bc_xy", C.c_int), ("bc_z", C.c_int), ("max_levels", C.c_int), ("no_symmetry", C.c_int),
                ("kernel_flags", C.c_int)]


class _TvParams(C.Structure):
    _fields_ = [("eps_delta", C.c_double), ("max_inner", C.c_int), ("max_backtracks", C.c_int),
                ("armijo_c", C.c_double), ("shrink_alpha", C.c_double), ("rel_tol", C.c_double)]


class _TvReport(C.Structure):
    _fields_ = [("inner_iters", C.c_int), ("trials", C.c_int), ("e_first", C.c_double), ("e_last", C.c_double)]


class _FbsParams(C.Structure):
    _fields_ = [("tv_weight", C.c_double), ("step", C.c_double), ("n_levels", C.c_int),
                ("iters_per_level", C.POINTER(C.c_int)), ("nonneg", C.c_int), ("use_initial", C.c_int),
                ("backprojector", C.c_int), ("conv_tol", C.c_double), ("tv", _TvParams)]


class _FbsReport(C.Structure):
    _fields_ = [("n_iters_total", C.c_int), ("objective", C.POINTER(C.c_double)),
                ("step_abs", C.POINTER(C.c_double)), ("iters_done", C.POINTER(C.c_int)), ("inner_total", C.c_int), ("trials_total", C.c_int),
                ("ms_total", C.c_float)]


_BCAST_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_ulonglong, C.c_int, C.c_void_p)
_ALLRED_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_ulonglong, C.c_void_p)


class _Comm(C.Structure):
    _fields_ = [("rank", C.c_int), ("world", C.c_int), ("ctx", C.c_void_p), ("broadcast", _BCAST_FN),
                ("allreduce_sum_f64", _ALLRED_FN)]


@dataclass
class TvReport:
    inner_iters: int
    trials: int
    e_first: float
    e_last: float


@dataclass
class FbsReport:
    n_iters_total: int
    objective: np.ndarray
    step_abs: np.ndarray
    inner_total: int
    trials_total: int
    ms_total: float
    iters_done: tuple = ()


_lib = None


def library_path() -> str:
    return _build.LIB


def load_library():
    """dlopen libcbct.so (building it with nvcc first if it is missing) and type its entry points."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_build.LIB):
        _build.build()
    lib = C.CDLL(_build.LIB)
    vp, ip, dp = C.c_void_p, C.c_int, C.c_double
    lib.cbct_geometry_create.argtypes = [C.POINTER(_Desc), C.POINTER(vp)]
    lib.cbct_geometry_destroy.argtypes = [vp]
    lib.cbct_geometry_destroy.restype = None
    lib.cbct_geometry_symmetry.argtypes = [vp, ip]
    lib.cbct_geometry_back_path.argtypes = [vp, ip]
    lib.cbct_bound_violations.argtypes = [vp, C.POINTER(C.c_uint), vp]
    lib.cbct_geometry_device_bytes.argtypes = [vp]
    lib.cbct_geometry_device_bytes.restype = C.c_ulonglong
    lib.cbct_forward_project.argtypes = [vp, ip, vp, vp, vp]
    lib.cbct_back_project.argtypes = [vp, ip, vp, vp, vp]
    lib.cbct_back_project_eq6.argtypes = [vp, ip, vp, vp, vp]
    lib.cbct_count_samples.argtypes = [vp, ip, C.POINTER(C.c_ulonglong), vp]
    lib.cbct_step_bound.argtypes = [vp, ip, C.POINTER(dp), vp]
    lib.cbct_quality_metrics.argtypes = [vp, ip, vp, vp, C.POINTER(dp), C.POINTER(dp), vp]
    lib.cbct_quality_metrics_static.argtypes = [vp, vp, C.c_ulonglong, vp, vp]
    lib.cbct_tv_prox.argtypes = [vp, ip, vp, vp, dp, ip, C.POINTER(_TvParams), C.POINTER(_TvReport), vp]
    lib.cbct_tv_energy.argtypes = [vp, ip, vp, dp, C.POINTER(dp), vp]
    lib.cbct_restrict_volume.argtypes = [vp, ip, vp, vp, vp]
    lib.cbct_bin_projections.argtypes = [vp, ip, vp, vp, vp]
    lib.cbct_prolong_volume.argtypes = [vp, ip, vp, vp, vp]
    lib.cbct_fbs_reconstruct.argtypes = [vp, vp, vp, C.POINTER(_FbsParams), C.POINTER(_FbsReport), vp]
    lib.cbct_fbs_reconstruct_host.argtypes = [vp, vp, vp, C.POINTER(_FbsParams), C.POINTER(_FbsReport), vp]
    lib.cbct_fbs_reconstruct_sharded.argtypes = [vp, C.POINTER(_Comm), vp, vp, C.POINTER(_FbsParams), C.POINTER(_FbsReport), vp]
    lib.cbct_shard_range.argtypes = [ip, ip, ip, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    lib.cbct_shard_units.argtypes = [vp, ip, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]
    lib.cbct_launch_count.argtypes = [vp]
    lib.cbct_launch_count.restype = C.c_ulonglong
    lib.cbct_set_stage_timing.argtypes = [vp, ip]
    lib.cbct_get_stage_ms.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_ulonglong)]
    lib.cbct_gather_ceiling.argtypes = [vp, C.c_ulonglong, ip, ip, ip, vp, C.POINTER(C.c_float), C.POINTER(C.c_ulonglong), vp]
    lib.cbct_last_error.restype = C.c_char_p
    lib.cbct_version.restype = C.c_char_p
    for name in EXPORTS:
        getattr(lib, name)          # AttributeError here = a declared symbol is not exported
    _lib = lib
    return lib


def _check(status: int):
    if status != CBCT_OK:
        raise CbctError(status, load_library().cbct_last_error().decode())


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dev(t, n: int, name: str):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{name}: need a contiguous float32 CUDA tensor")
    if t.numel() != n:
        raise ValueError(f"{name}: {t.numel()} elements, expected {n}")
    return C.c_void_p(t.data_ptr())


def _tv_params(fbs) -> _TvParams:
    return _TvParams(fbs.eps_delta, fbs.max_inner, fbs.max_backtracks, fbs.armijo_c, fbs.shrink_alpha, fbs.rel_tol)


class Geometry:
    """Owning wrapper of a `cbct_geometry*` handle (cbct_geometry_create / _destroy).

    `desc` is any object with the attributes of `inputs.Geometry`.
    """

    def __init__(self, desc, max_levels: int = 1, no_symmetry: bool = False, no_tma: bool = False, host_armijo: bool = False,
                 tv_scalar_tiles: bool = False, back_lists_on_the_fly: bool = False, no_reflection: bool = False,
                 no_fold: bool = False):
        lib = load_library()
        self._h = C.c_void_p()
        self.desc = desc
        self.max_levels = int(max_levels)
        d = _Desc()
        d.nx, d.ny, d.nz = desc.nx, desc.ny, desc.nz
        d.hx, d.hy, d.hz = desc.hx, desc.hy, desc.hz
        for a in range(3):
            d.vol_off[a] = float(desc.vol_off[a])
        d.nu, d.nv, d.du, d.dv = desc.nu, desc.nv, desc.du, desc.dv
        d.det_off_u, d.det_off_v = desc.det_off_u, desc.det_off_v
        d.sad, d.sdd, d.n_proj = desc.sad, desc.sdd, desc.n_proj
        ang = np.ascontiguousarray(desc.angles_rad(), dtype=np.float64)
        d.angles_rad = ang.ctypes.data_as(C.POINTER(C.c_double))
        d.bc_xy, d.bc_z, d.max_levels = desc.bc_xy, desc.bc_z, self.max_levels
        d.no_symmetry = int(bool(no_symmetry))
        # CBCT_KERNEL_NO_TMA | CBCT_KERNEL_HOST_ARMIJO | CBCT_KERNEL_TV_SCALAR_TILES | CBCT_KERNEL_BACK_LISTS_ON_THE_FLY
        d.kernel_flags = ((1 if no_tma else 0) | (2 if host_armijo else 0) | (4 if tv_scalar_tiles else 0) |
                          (8 if back_lists_on_the_fly else 0) | (16 if no_reflection else 0) |   # ... | CBCT_KERNEL_NO_REFLECTION
                          (32 if no_fold else 0))                                                # | CBCT_KERNEL_NO_FOLD
        _check(lib.cbct_geometry_create(C.byref(d), C.byref(self._h)))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load_library().cbct_geometry_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # sizes ------------------------------------------------------------------
    def vol_shape(self, level: int = 0):
        f = 1 << level
        return (self.desc.nz // f, self.desc.ny // f, self.desc.nx // f)

    def proj_shape(self, level: int = 0):
        f = 1 << level
        return (self.desc.n_proj, self.desc.nv // f, self.desc.nu // f)

    def _nvox(self, level):
        return int(np.prod(self.vol_shape(level)))

    def _nray(self, level):
        return int(np.prod(self.proj_shape(level)))

    @property
    def symmetry(self) -> int:
        return int(load_library().cbct_geometry_symmetry(self._h, 0))

    def back_path(self, level: int = 0) -> str:
        """cbct_geometry_back_path: which exact-transpose back-projector the level runs."""
        return {0: "gather", 1: "list", 2: "tma"}[int(load_library().cbct_geometry_back_path(self._h, level))]

    def bound_violations(self, stream=None) -> int:
        n = C.c_uint(0)
        _check(load_library().cbct_bound_violations(self._h, C.byref(n), _stream_ptr(stream)))
        return int(n.value)

    @property
    def device_bytes(self) -> int:
        return int(load_library().cbct_geometry_device_bytes(self._h))

    @property
    def launch_count(self) -> int:
        return int(load_library().cbct_launch_count(self._h))

    # operators --------------------------------------------------------------
    def forward_project(self, vol, proj, level: int = 0, stream=None):
        _check(load_library().cbct_forward_project(self._h, level, _dev(vol, self._nvox(level), "vol"),
                                                   _dev(proj, self._nray(level), "proj"), _stream_ptr(stream)))
        return proj

    def back_project(self, proj, vol, level: int = 0, stream=None):
        _check(load_library().cbct_back_project(self._h, level, _dev(proj, self._nray(level), "proj"),
                                                _dev(vol, self._nvox(level), "vol"), _stream_ptr(stream)))
        return vol

    def back_project_eq6(self, proj, vol, level: int = 0, stream=None):
        _check(load_library().cbct_back_project_eq6(self._h, level, _dev(proj, self._nray(level), "proj"),
                                                    _dev(vol, self._nvox(level), "vol"), _stream_ptr(stream)))
        return vol

    def count_samples(self, level: int = 0, stream=None) -> int:
        out = C.c_ulonglong()
        _check(load_library().cbct_count_samples(self._h, level, C.byref(out), _stream_ptr(stream)))
        return int(out.value)

    def step_bound(self, level: int = 0, stream=None) -> float:
        out = C.c_double()
        _check(load_library().cbct_step_bound(self._h, level, C.byref(out), _stream_ptr(stream)))
        return out.value

    def tv_prox(self, g, f, weight_w: float, fbs, nonneg: bool = False, level: int = 0, report: bool = True,
                stream=None):
        tp = _tv_params(fbs)
        rep = _TvReport()
        _check(load_library().cbct_tv_prox(self._h, level, _dev(g, self._nvox(level), "g"),
                                           _dev(f, self._nvox(level), "f"), C.c_double(weight_w), int(bool(nonneg)),
                                           C.byref(tp), C.byref(rep) if report else None, _stream_ptr(stream)))
        return TvReport(rep.inner_iters, rep.trials, rep.e_first, rep.e_last) if report else None

    def tv_energy(self, f, eps_delta: float, level: int = 0, stream=None) -> float:
        out = C.c_double()
        _check(load_library().cbct_tv_energy(self._h, level, _dev(f, self._nvox(level), "f"),
                                             C.c_double(eps_delta), C.byref(out), _stream_ptr(stream)))
        return out.value

    def quality_metrics(self, f, f0, level: int = 0, stream=None):
        """(relative error e, correlation coefficient c) of f against the ground truth f0."""
        e, c = C.c_double(), C.c_double()
        _check(load_library().cbct_quality_metrics(self._h, level, _dev(f, self._nvox(level), "f"),
                                                   _dev(f0, self._nvox(level), "f0"), C.byref(e), C.byref(c),
                                                   _stream_ptr(stream)))
        return e.value, c.value

    def restrict_volume(self, fine, coarse, level: int = 0, stream=None):
        _check(load_library().cbct_restrict_volume(self._h, level, _dev(fine, self._nvox(level), "fine"),
                                                   _dev(coarse, self._nvox(level + 1), "coarse"), _stream_ptr(stream)))
        return coarse

    def bin_projections(self, fine, coarse, level: int = 0, stream=None):
        _check(load_library().cbct_bin_projections(self._h, level, _dev(fine, self._nray(level), "fine"),
                                                   _dev(coarse, self._nray(level + 1), "coarse"), _stream_ptr(stream)))
        return coarse

    def prolong_volume(self, coarse, fine, level: int = 0, stream=None):
        _check(load_library().cbct_prolong_volume(self._h, level, _dev(coarse, self._nvox(level + 1), "coarse"),
                                                  _dev(fine, self._nvox(level), "fine"), _stream_ptr(stream)))
        return fine

    # reconstruction ---------------------------------------------------------
    def _fbs_args(self, fbs, use_initial, want_objective):
        iters = np.ascontiguousarray(fbs.iters_per_level, dtype=np.int32)
        p = _FbsParams()
        p.tv_weight, p.step, p.n_levels = fbs.tv_weight, fbs.step, len(iters)
        p.iters_per_level = iters.ctypes.data_as(C.POINTER(C.c_int))
        p.nonneg, p.use_initial = int(bool(fbs.nonneg)), int(bool(use_initial))
        p.backprojector = int(getattr(fbs, "backprojector", 0))
        p.conv_tol = float(getattr(fbs, "conv_tol", 0.0))
        p.tv = _tv_params(fbs)
        obj = np.zeros(int(iters.sum()) if want_objective else 0)
        step_abs = np.zeros(len(iters))
        done = np.zeros(len(iters), dtype=np.int32)
        r = _FbsReport()
        r.iters_done = done.ctypes.data_as(C.POINTER(C.c_int))
        r.objective = obj.ctypes.data_as(C.POINTER(C.c_double)) if want_objective else None
        r.step_abs = step_abs.ctypes.data_as(C.POINTER(C.c_double))
        return p, r, (iters, obj, step_abs, done)

    @staticmethod
    def _fbs_report(r, keep):
        _, obj, step_abs, done = keep
        return FbsReport(r.n_iters_total, obj[:int(done.sum())] if len(obj) else obj, step_abs, r.inner_total,
                         r.trials_total, float(r.ms_total), tuple(int(x) for x in done))

    def fbs_reconstruct(self, proj_y, vol_inout, fbs, use_initial: bool = False, objective: bool = True,
                        stream=None) -> FbsReport:
        """cbct_fbs_reconstruct on device tensors (finest-level sizes)."""
        p, r, keep = self._fbs_args(fbs, use_initial, objective)
        _check(load_library().cbct_fbs_reconstruct(self._h, _dev(proj_y, self._nray(0), "proj_y"),
                                                   _dev(vol_inout, self._nvox(0), "vol_inout"), C.byref(p),
                                                   C.byref(r), _stream_ptr(stream)))
        return self._fbs_report(r, keep)

    def fbs_reconstruct_host(self, proj_y, vol_inout, fbs, use_initial: bool = False, objective: bool = False,
                             stream=None) -> FbsReport:
        """cbct_fbs_reconstruct_host on HOST float32 buffers (numpy arrays or CPU tensors, ideally pinned)."""
        def host_ptr(x, n, name):
            import torch
            if isinstance(x, torch.Tensor):
                if x.is_cuda or x.dtype != torch.float32 or not x.is_contiguous() or x.numel() != n:
                    raise TypeError(f"{name}: need a contiguous float32 CPU tensor of {n} elements")
                return C.c_void_p(x.data_ptr())
            if not (isinstance(x, np.ndarray) and x.dtype == np.float32 and x.flags.c_contiguous and x.size == n):
                raise TypeError(f"{name}: need a contiguous float32 array of {n} elements")
            return C.c_void_p(x.ctypes.data)
        p, r, keep = self._fbs_args(fbs, use_initial, objective)
        _check(load_library().cbct_fbs_reconstruct_host(self._h, host_ptr(proj_y, self._nray(0), "proj_y"),
                                                        host_ptr(vol_inout, self._nvox(0), "vol_inout"), C.byref(p),
                                                        C.byref(r), _stream_ptr(stream)))
        return self._fbs_report(r, keep)

    def fbs_reconstruct_sharded(self, comm: "Comm", proj_y, vol_inout, fbs, use_initial: bool = False,
                                objective: bool = True, stream=None) -> FbsReport:
        """cbct_fbs_reconstruct_sharded: this rank's part of a reconstruction sharded over comm.world GPUs."""
        p, r, keep = self._fbs_args(fbs, use_initial, objective)
        _check(load_library().cbct_fbs_reconstruct_sharded(self._h, C.byref(comm.struct), _dev(proj_y, self._nray(0), "proj_y"),
                                                           _dev(vol_inout, self._nvox(0), "vol_inout"), C.byref(p),
                                                           C.byref(r), _stream_ptr(stream)))
        if comm.error is not None:
            raise comm.error
        return self._fbs_report(r, keep)

    def shard_units(self, level: int = 0):
        """(base views, z-units, slices per z-unit) the level's projectors are sharded in."""
        a, b, c = C.c_int(0), C.c_int(0), C.c_int(0)
        _check(load_library().cbct_shard_units(self._h, level, C.byref(a), C.byref(b), C.byref(c)))
        return a.value, b.value, c.value

    # profiling --------------------------------------------------------------
    def set_stage_timing(self, enable: bool):
        _check(load_library().cbct_set_stage_timing(self._h, int(bool(enable))))

    STAGES = ("transpose", "forward", "back", "tv_grad", "tv_trial", "tv_update", "reduce", "transfer")

    def stage_ms(self):
        """{stage: (milliseconds, launch groups)} accumulated since set_stage_timing."""
        ms = (C.c_float * len(self.STAGES))()
        calls = (C.c_ulonglong * len(self.STAGES))()
        _check(load_library().cbct_get_stage_ms(self._h, ms, calls))
        return {k: (float(m), int(c)) for k, m, c in zip(self.STAGES, ms, calls)}


def shard_range(n_units: int, world: int, rank: int):
    """cbct_shard_range: the contiguous share [lo, hi) of `rank` (pure host arithmetic, no device needed)."""
    lo, hi = C.c_int(0), C.c_int(0)
    _check(load_library().cbct_shard_range(n_units, world, rank, C.byref(lo), C.byref(hi)))
    return lo.value, hi.value


class _DevBytes:
    """A window of device memory as a __cuda_array_interface__ object (zero copy into a torch tensor)."""

    def __init__(self, ptr: int, n: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": typestr, "data": (ptr, False), "version": 2}


def device_window(ptr: int, n: int, typestr: str = "|u1"):
    import torch
    return torch.as_tensor(_DevBytes(ptr, n, typestr), device="cuda")


class Comm:
    """cbct_comm: the two collectives of cbct_fbs_reconstruct_sharded as Python callables on torch tensors that alias the
    handle's device memory.  `broadcast(tensor_u8, root)` and `allreduce_sum(tensor_f64)` work in place and must be ordered
    on the torch stream current when they are called (the binding makes the library's stream current around each call)."""

    def __init__(self, rank: int, world: int, broadcast, allreduce_sum):
        import torch
        self.error = None

        def on_stream(stream_ptr):
            return torch.cuda.stream(torch.cuda.ExternalStream(stream_ptr or 0))

        def bcast(_ctx, ptr, nbytes, root, stream_ptr):
            try:
                with on_stream(stream_ptr):
                    broadcast(device_window(ptr, nbytes), root)
                return 0
            except Exception as e:      # nothing may propagate through the C frames
                self.error = e
                return 1

        def allred(_ctx, ptr, n, stream_ptr):
            try:
                with on_stream(stream_ptr):
                    allreduce_sum(device_window(ptr, n, "<f8"))
                return 0
            except Exception as e:
                self.error = e
                return 1

        self._keep = (_BCAST_FN(bcast), _ALLRED_FN(allred))
        self.struct = _Comm(rank, world, None, self._keep[0], self._keep[1])
        self.rank, self.world = rank, world


def torch_distributed_comm(group=None) -> Comm:
    """The communicator over a torch.distributed process group (backend nccl: one process per GPU)."""
    import torch.distributed as dist
    ranks = dist.get_process_group_ranks(group) if group is not None else list(range(dist.get_world_size()))

    def broadcast(t, root):
        dist.broadcast(t, src=ranks[root], group=group)

    def allreduce_sum(t):
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)

    return Comm(dist.get_rank(group), dist.get_world_size(group), broadcast, allreduce_sum)


def gather_ceiling(buf, variant: int, reuse: int = 1, iters: int = 64, stream=None):
    """cbct_gather_ceiling: (GB/s the lanes were served, milliseconds) of one calibration launch over `buf`."""
    import torch
    if not (isinstance(buf, torch.Tensor) and buf.is_cuda and buf.dtype == torch.float32 and buf.is_contiguous()):
        raise TypeError("buf: need a contiguous float32 CUDA tensor")
    sink = torch.zeros(1, device=buf.device, dtype=torch.float32)
    ms, nbytes = C.c_float(0.0), C.c_ulonglong(0)
    _check(load_library().cbct_gather_ceiling(C.c_void_p(buf.data_ptr()), buf.numel(), variant, reuse, iters,
                                              C.c_void_p(sink.data_ptr()), C.byref(ms), C.byref(nbytes), _stream_ptr(stream)))
    return nbytes.value / (ms.value * 1e-3) / 1e9, ms.value


def geometry_create(desc, max_levels: int = 1, no_symmetry: bool = False, no_tma: bool = False,
                    host_armijo: bool = False, tv_scalar_tiles: bool = False, back_lists_on_the_fly: bool = False,
                    no_reflection: bool = False, no_fold: bool = False) -> Geometry:
    return Geometry(desc, max_levels, no_symmetry, no_tma, host_armijo, tv_scalar_tiles, back_lists_on_the_fly, no_reflection,
                    no_fold)


STATIC_MAX_ELEMS = 1 << 28      # CBCT_STATIC_MAX_ELEMS


def quality_metrics_static(f, f0, out2, stream=None, n: int | None = None):
    """cbct_quality_metrics_static: (e, c) of f against f0 into the 2-element float64 CUDA tensor `out2`, asynchronously on the
    stream; no geometry handle, no allocation (the scratch is a static __device__ array inside the library, shared by all
    calls: do not overlap them).  `n` (default: all elements of f) may not exceed STATIC_MAX_ELEMS."""
    import torch
    n = f.numel() if n is None else int(n)
    if not (isinstance(out2, torch.Tensor) and out2.is_cuda and out2.dtype == torch.float64 and out2.is_contiguous()
            and out2.numel() == 2):
        raise TypeError("out2: need a contiguous float64 CUDA tensor of 2 elements")
    for name, t in (("f", f), ("f0", f0)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
            raise TypeError(f"{name}: need a contiguous float32 CUDA tensor")
        if n <= STATIC_MAX_ELEMS and t.numel() < n:        # beyond the maximum the library refuses before it reads anything
            raise ValueError(f"{name}: {t.numel()} elements, fewer than n = {n}")
    _check(load_library().cbct_quality_metrics_static(C.c_void_p(f.data_ptr()), C.c_void_p(f0.data_ptr()), C.c_ulonglong(n),
                                                      C.c_void_p(out2.data_ptr()), _stream_ptr(stream)))
    return out2


def version() -> str:
    return load_library().cbct_version().decode()
