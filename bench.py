#!/usr/bin/env python
"""bench.py -- FBS iterations/s of the CUDA path on BASELINE.json's metric configuration.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload config3]

One "step" = one pass of the whole hot path (SURVEY.md section 8(a) rows A1-A7, A9's E2): one
finest-level forward-backward-splitting iteration -- forward projection + residual + E2,
exact-transpose back-projection + gradient step, TV-prox (Armijo gradient descent), clip -- on
config 3 of BASELINE.json (256^3 volume, 40 views of 512x384; synthetic torso phantom, Poisson
noise), started from the volume the two coarser multi-grid levels hand to the finest one.
The multi-grid driver (A8) is timed as the full reconstruction ("recon_seconds").

Prints ONE JSON line (rank 0).  Under torchrun every rank reconstructs its own independent problem
(same geometry, own noise seed): no data-path collective, "scaling": "weak".

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1001_0599_b200 import inputs as I  # noqa: E402

METRIC = "fbs_iterations_per_second"
UNIT = "iter/s"

COUNTERS_FILE = os.path.join(ROOT, "profiles", "r02_counters.json")


def _load_counters():
    """ncu counters per kernel of the FBS step (DRAM bytes per launch, L1 / L2 hit rates, ...) from the tracked record the
    capture step wrote (`python -m paper_1001_0599_b200.ncu_counters`): evidence for each kernel's memory path, not a timing.
    The record carries a hash of the kernel sources it was captured from; when the sources have changed since, the
    counters are stale and are NOT quoted (roofline.traffic = null)."""
    from paper_1001_0599_b200 import ncu_counters
    if not os.path.exists(COUNTERS_FILE):
        return {}, {"counters_file": None}
    rec = json.load(open(COUNTERS_FILE))
    fresh = rec.get("kernel_sources_sha256") == ncu_counters.kernel_sources_sha256()
    meta = {"counters_file": os.path.relpath(COUNTERS_FILE, ROOT), "counters_commit": rec.get("counters_commit"),
            "counters_match_kernel_sources": fresh}
    return (rec.get("kernels", {}) if fresh else {}), meta


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.lines, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def __exit__(self, *exc):
        if self.proc is not None:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
            self.thread.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.lines:
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for n, v in zip(names, parts[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "samples": len(sm)}


def rank_env():
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) when launched plainly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def rank_seed(seed: int, rank: int) -> int:
    """Every rank reconstructs its own problem: same phantom and geometry, own noise realisation."""
    return seed + 1000 * rank


def max_over_ranks(ms: float, world: int, device="cuda") -> float:
    """Device time of the slowest rank (the job's time); a no-op for one process."""
    if world == 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(steps: int, world: int, ms_total: float) -> float:
    """Whole-job throughput: every rank did `steps` units in `ms_total` (max over ranks)."""
    return world * steps / (ms_total / 1e3)


def fov_mask(g) -> np.ndarray:
    """Voxels whose centre every view sees: (u*, v*) of Eq. A6 inside the detector for all angles.
    Measurement-side helper for the error restricted to the field of view (reading R4)."""
    x = (np.arange(g.nx) - 0.5 * (g.nx - 1)) * g.hx + g.vol_off[0]
    yy = (np.arange(g.ny) - 0.5 * (g.ny - 1)) * g.hy + g.vol_off[1]
    z = (np.arange(g.nz) - 0.5 * (g.nz - 1)) * g.hz + g.vol_off[2]
    umax, vmax = 0.5 * g.nu * g.du, 0.5 * g.nv * g.dv
    inplane = np.ones((g.ny, g.nx), dtype=bool)
    mag_min = np.full((g.ny, g.nx), np.inf)
    X, Y = np.meshgrid(x, yy)
    for t in g.angles_rad():
        c, s_ = np.cos(t), np.sin(t)
        rn = X * c + Y * s_ + g.sad
        u = g.sdd * (X * s_ - Y * c) / rn
        inplane &= np.abs(u - g.det_off_u) <= umax
        mag_min = np.minimum(mag_min, rn / g.sdd)          # |z| <= vmax rn / sdd for the view that sees least of the column
    zlim = vmax * mag_min                                       # (det_off_v = 0 in every config)
    return inplane[None, :, :] & (np.abs(z)[:, None, None] <= zlim[None, :, :])


def workload(name: str):
    k = {"config1": 1, "config2": 2, "config3": 3, "config4": 4}[name]
    cfg = I.config(k)
    return k, cfg


# ---------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline of our arm; the whole of --impl reference)
# ---------------------------------------------------------------------------------------------

def oracle_sample(cfg, y, views: int, z_div: int):
    """The oracle's cost of one finest-level FBS iteration, from a bounded sample at FULL resolution:
    P and P^T on `views` of the workload's views (their cost is a sum over views, so the full
    operator is n_proj/views times the sample) and one TV-prox call on a slab of nz/z_div slices
    of g = f - tau c_norm P^T(P f - y) built from those views (full call = z_div times the slab)."""
    from oracle import cbct_oracle as orc
    orc.build()
    g = cfg.geom
    sel = (np.arange(views) * g.n_proj // views + g.n_proj // (2 * views)) % g.n_proj
    gs = g.replace(n_proj=views, angles=g.angles_rad()[sel])
    f = I.paint(cfg.ellipsoids, g).astype(np.float64) * 0.9
    t0 = time.perf_counter()
    T = orc.forward(gs, f) - y[sel]
    t1 = time.perf_counter()
    b = orc.back(gs, T)
    t2 = time.perf_counter()
    c_norm = 2.0 * f.size / T.size
    tau = cfg.fbs.step / (c_norm * 2.0e5 * views / g.n_proj)      # order of magnitude of 1/Lhat; timing only
    nzs = max(4, g.nz // z_div)
    k0 = (g.nz - nzs) // 2
    gz = g.replace(nz=nzs)
    gg = (f - tau * c_norm * b)[k0:k0 + nzs]
    t3 = time.perf_counter()
    _, rep = orc.tv_prox(gz, gg, tau * cfg.fbs.tv_weight, cfg.fbs)
    t4 = time.perf_counter()
    sec_full = (t1 - t0) * g.n_proj / views + (t2 - t1) * g.n_proj / views + (t4 - t3) * g.nz / nzs
    return {"seconds_full_iteration": sec_full, "sample_seconds": t4 - t0 - (t3 - t2), "threads": orc.threads(),
            "parts_s": {"P": (t1 - t0) * g.n_proj / views, "PT": (t2 - t1) * g.n_proj / views,
                        "tv_prox": (t4 - t3) * g.nz / nzs, "tv_inner": rep.inner_iters},
            "sample": f"oracle P and P^T on {views} of {g.n_proj} views at full resolution ({g.nx}x{g.ny}x{g.nz}, "
                      f"{g.nu}x{g.nv}) scaled x{g.n_proj / views:.4g}, plus one oracle TV-prox call on a "
                      f"{nzs}-slice slab scaled x{g.nz / nzs:.4g}; sum = one finest-level FBS iteration"}


def cpu_baseline(cfg, y, budget: str = "default"):
    # the sample is sized for ~10 s of oracle work on the GPU box's host (all 40 views of config 3); "small" (the per-step
    # sample of the reference arm, repeated warmup + steps times) is 16 views and a sixteenth of the TV slab, ~4 s
    g = cfg.geom
    cost = float(g.nu) * g.nv * max(g.nx, g.ny)                     # per-view cost of P / P^T, relative
    views = min(g.n_proj, max(1, int(round(40 * 5.0e7 / cost))))
    z_div = 1 if g.nx * g.ny * g.nz <= 2.0e7 else 4
    if budget != "default":
        # the oracle's back-projector deals views to threads: fewer views than threads would idle cores
        views, z_div = min(g.n_proj, max(1, int(round(16 * 5.0e7 / cost)))), 16
    r = oracle_sample(cfg, y, views, z_div)
    return {"value": 1.0 / r["seconds_full_iteration"], "unit": UNIT, "cores": r["threads"], "kind": "oracle",
            "sample": r["sample"], "sample_seconds": round(r["sample_seconds"], 3),
            "full_iteration_seconds_by_part": {k: round(v, 3) for k, v in r["parts_s"].items()},
            "extrapolated": not (views == g.n_proj and z_div == 1)}


def run_reference(args):
    rank, _, _ = rank_env()
    if rank != 0:
        return
    k, cfg = workload(args.workload)
    y = I.make_projections(cfg)
    times = []
    base = None
    for i in range(args.warmup + args.steps):
        base = cpu_baseline(cfg, y, "small")
        if i >= args.warmup:
            times.append(1.0 / base["value"])
    sec = float(np.mean(times))
    g = cfg.geom
    line = {"impl": "reference", "metric": METRIC, "value": 1.0 / sec, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config{k}: {g.nx}x{g.ny}x{g.nz} voxels, {g.n_proj} views of {g.nu}x{g.nv}, "
                                   "one finest-level FBS iteration (scaled up from a bounded full-resolution sample)"},
            "cpu_baseline": {"value": 1.0 / sec, "unit": UNIT, "kind": "oracle", "cores": base["cores"],
                             "sample": base["sample"]},
            "e2e": {"value": 1.0 / sec, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------

def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1001_0599_b200 import cbct

    rank, world, local = rank_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    hbm_peak, sm_max_mhz, peak_src = _peaks()

    k, cfg = workload(args.workload)
    g = cfg.geom
    sharded = bool(args.sharded)
    if not sharded:
        cfg.seed = rank_seed(cfg.seed, rank)        # replicas: every rank its own noise realisation
    y_host = I.make_projections(cfg)                # sharded: ONE problem, the same data on every rank
    n_levels = len(cfg.fbs.iters_per_level)
    fbs = cfg.fbs
    stream = torch.cuda.Stream()
    nvox, nray = int(np.prod(g.vol_shape)), int(np.prod(g.proj_shape))

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    with torch.cuda.stream(stream), cbct.geometry_create(g, max_levels=n_levels) as h:
        y = torch.from_numpy(y_host).cuda()
        f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        one = I.FbsSetup(**{**fbs.__dict__, "iters_per_level": (1,)})

        # the volume the coarser levels hand to the finest level (untimed set-up)
        if n_levels > 1:
            pre = I.FbsSetup(**{**fbs.__dict__, "iters_per_level": tuple(fbs.iters_per_level[:-1]) + (0,)})
            h.fbs_reconstruct(y, f, pre, objective=False)
        S = h.count_samples()
        h.step_bound()
        f_start = f.clone()
        back_path = h.back_path(0)

        # ---- measured gather ceilings: the calibration kernel over a buffer the size of the staged
        # volume copy, each pattern from L2 (every run new to the SM) and from L1 (a 16 KB tile re-read 256 times), and the
        # shared-memory patterns of the TMA back-projector
        cal = torch.rand(70 * 2 ** 20 // 4, device="cuda")
        ceilings = {}
        for key, variant, reuse, iters in (("ldg4_run128B_from_l2", 0, 1, 128), ("ldg4_run128B_from_l1", 0, 256, 256),
                                           ("ldg16_stride2_from_l2", 1, 1, 64), ("ldg16_stride2_from_l1", 1, 256, 128),
                                           ("lds16_stride2_plain", 2, 1, 512), ("lds16_stride2_parity_split", 3, 1, 512)):
            ceilings[key] = max(cbct.gather_ceiling(cal, variant, reuse, iters, stream=stream)[0] for _ in range(3))
        del cal

        # --sharded (NEXT-4): the ranks reconstruct ONE problem, the projectors sharded by output ownership
        # (cbct_fbs_reconstruct_sharded; strong scaling).  At one GPU the communicator is trivial.
        comm = None
        if sharded:
            comm = (cbct.torch_distributed_comm() if world > 1 else
                    cbct.Comm(0, 1, lambda t, root: None, lambda t: None))

        def run_fbs(setup, **kw):
            if comm is not None:
                return h.fbs_reconstruct_sharded(comm, y, f, setup, stream=stream, **kw)
            return h.fbs_reconstruct(y, f, setup, stream=stream, **kw)

        def step_device():
            return run_fbs(one, use_initial=True, objective=False)

        for _ in range(args.warmup):
            step_device()
        # ---- K steps as K separate one-iteration calls: per-step statistics ----------------------
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
        barrier()
        ev0.record(stream)
        for i_step in range(args.steps):
            step_device()
            marks[i_step].record(stream)
        barrier()
        per_step = [a_.elapsed_time(b_) for a_, b_ in zip([ev0] + marks[:-1], marks)]
        # ---- timed region: EXACTLY K steps = one cbct_fbs_reconstruct call of K finest-level iterations -----------
        # (the library's own loop: inside one call the next iteration's forward projection is queued while the host
        # reads the TV trial's sums, which K separate calls cannot do)
        k_steps = I.FbsSetup(**{**fbs.__dict__, "iters_per_level": (args.steps,)})
        f.copy_(f_start)
        l0 = h.launch_count
        barrier()
        with ClockSampler(local) as clk:
            torch.cuda.profiler.start()        # cudaProfilerStart: `ncu --profile-from-start off` sees only the timed region
            ev0.record(stream)
            r = run_fbs(k_steps, use_initial=True, objective=False)
            ev1.record(stream)
            barrier()
            torch.cuda.profiler.stop()
        inner, trials = r.inner_total, r.trials_total
        ms_total = max_over_ranks(ev0.elapsed_time(ev1), world)
        launches = h.launch_count - l0
        clocks = clk.summary()

        # ---- e2e: the same step through the HOST entry point, copies inside the timed region -
        y_pin = torch.from_numpy(y_host).pin_memory()
        f_pin = f.cpu().pin_memory()
        def step_e2e():
            if comm is None:
                h.fbs_reconstruct_host(y_pin, f_pin, one, use_initial=True, stream=stream)
            else:           # no host entry point of the sharded call: the same copies, issued here
                y.copy_(y_pin, non_blocking=True)
                f.copy_(f_pin, non_blocking=True)
                run_fbs(one, use_initial=True, objective=False)
                f_pin.copy_(f, non_blocking=True)
                stream.synchronize()

        for _ in range(max(1, min(args.warmup, 2))):
            step_e2e()
        barrier()
        ev0.record(stream)
        for _ in range(args.steps):
            step_e2e()
        ev1.record(stream)
        barrier()
        ms_e2e = max_over_ranks(ev0.elapsed_time(ev1), world)

        # ---- per-kernel attribution (CUDA events on the library's stream, synchronising) ----
        f.copy_(f_start)
        h.set_stage_timing(True)
        for _ in range(args.steps):
            step_device()
        stages = h.stage_ms()
        h.set_stage_timing(False)

        # ---- whole reconstruction: all levels, all iterations (rank 0 reports) ---------------
        recon = None
        recon_extra = {}
        if not args.no_recon:
            f.zero_()
            barrier()
            rr = run_fbs(fbs, objective=False)
            e_rec, c_rec = h.quality_metrics(f, torch.from_numpy(I.paint(cfg.ellipsoids, g)).cuda(), stream=stream)
            t0 = time.perf_counter()
            vol_host = np.zeros(g.vol_shape, dtype=np.float32)
            hr = h.fbs_reconstruct_host(y_host, vol_host, fbs, stream=stream)
            wall = time.perf_counter() - t0
            truth = I.paint(cfg.ellipsoids, g)
            recon = {"recon_seconds": rr.ms_total / 1e3, "recon_seconds_host_buffers_wall": wall,
                     "iterations": int(rr.n_iters_total), "levels": n_levels,
                     "tv_inner_total": int(rr.inner_total), "tv_trials_total": int(rr.trials_total),
                     # the paper's Table 1 metrics (L263) of the reconstruction against the voxelised phantom
                     "rel_error_vs_phantom": e_rec, "correlation_vs_phantom": c_rec,
                     "rel_error_vs_phantom_host_entry": float(np.linalg.norm(vol_host - truth) / np.linalg.norm(truth))}
            del hr
            # ---- beside the headline: the error inside the field of view, and the regime where the TV step does work ----
            # (reading R4: under the normalisation S5 the configs' TV weight 0.01 is a very weak regulariser -- every
            # prox call is one accepted step.  A coarse scan of the weight finds the one with the lowest error against the
            # phantom; K finest-level iterations are then timed at that weight.  Reported, never the headline `value`.)
            recon_extra = {}
            if rank == 0 and not args.no_extra:
                mask = fov_mask(g)
                t_dev = torch.from_numpy(truth).cuda()
                m_dev = torch.from_numpy(mask).cuda()

                def errors(vol):
                    d2 = (vol - t_dev) ** 2
                    return (float(torch.sqrt(d2.sum() / (t_dev ** 2).sum())),
                            float(torch.sqrt(d2[m_dev].sum() / (t_dev[m_dev] ** 2).sum())))

                scan = []
                for lam in (fbs.tv_weight, 1.0, 10.0, 100.0, 1000.0, 10000.0):
                    sl = I.FbsSetup(**{**fbs.__dict__, "tv_weight": lam})
                    f.zero_()
                    rl = h.fbs_reconstruct(y, f, sl, objective=False, stream=stream)
                    e_all, e_fov = errors(f)
                    scan.append({"tv_weight": lam, "rel_error_vs_phantom": e_all, "rel_error_inside_fov": e_fov,
                                 "recon_seconds": rl.ms_total / 1e3, "tv_inner_total": int(rl.inner_total),
                                 "tv_trials_total": int(rl.trials_total)})
                best = min(scan, key=lambda r_: r_["rel_error_inside_fov"])
                sb = I.FbsSetup(**{**fbs.__dict__, "tv_weight": best["tv_weight"]})
                f.zero_()
                h.fbs_reconstruct(y, f, I.FbsSetup(**{**sb.__dict__, "iters_per_level": tuple(fbs.iters_per_level[:-1]) + (0,)}),
                                  objective=False, stream=stream)
                kb = I.FbsSetup(**{**sb.__dict__, "iters_per_level": (args.steps,)})
                h.fbs_reconstruct(y, f, kb, use_initial=True, objective=False, stream=stream)     # warm-up
                h.set_stage_timing(True)
                rb = h.fbs_reconstruct(y, f, kb, use_initial=True, objective=False, stream=stream)
                st_b = h.stage_ms()
                h.set_stage_timing(False)
                rb2 = h.fbs_reconstruct(y, f, kb, use_initial=True, objective=False, stream=stream)
                tv_ms = sum(st_b[n][0] for n in ("tv_grad", "tv_trial", "tv_update")) / args.steps
                all_ms = sum(v_[0] for v_ in st_b.values()) / args.steps
                recon_extra = {"fov_voxel_fraction": float(mask.mean()),
                               "rel_error_inside_fov": scan[0]["rel_error_inside_fov"],
                               "tv_weight_scan": scan,
                               "tv_active_regime": {"tv_weight": best["tv_weight"], "ms_per_step": rb2.ms_total / args.steps,
                                                    "tv_inner_per_step": rb.inner_total / args.steps,
                                                    "tv_trials_per_step": rb.trials_total / args.steps,
                                                    "tv_ms_per_step": tv_ms, "tv_share_of_step": tv_ms / all_ms,
                                                    "note": "config 3 at the TV weight with the lowest in-FOV error of the scan; "
                                                            "an extra row, not the headline"}}
                del t_dev, m_dev

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    if recon:
        recon.update(recon_extra)

    K = args.steps
    sec_step = ms_total / 1e3 / K
    per = {name: {"ms_per_step": ms / K, "launches_per_step": c / K, "ms_per_launch": (ms / c if c else None)}
           for name, (ms, c) in stages.items()}
    # kernel rooflines.
    # P and P^T: every ray-voxel sample must pull 4 bytes (a volume cell / a residual value) through an SM's L1
    # data path: the gather roofline is 128 B/clk/SM x 148 SMs x f_clk = 32 samples/clk/SM.  The TV passes stream
    # the volume arrays once: HBM roofline (measured copy bandwidth).
    l1_peak_gbs = 148 * 128 * sm_max_mhz * 1e6 / 1e9
    counters, counters_meta = _load_counters() if args.workload == "config3" else ({}, {"counters_file": None})
    # the measured ceiling of each projector's own pattern: the forward projector's 4-byte loads of contiguous runs served
    # from L1; the back-projector's 16-byte loads two entries apart, from shared memory (TMA path) or from L1 (list kernel)
    measured = {"forward": ("ldg4_run128B_from_l1", ceilings["ldg4_run128B_from_l1"]),
                "back": (("lds16_stride2_parity_split", ceilings["lds16_stride2_parity_split"]) if back_path == "tma"
                         else ("ldg16_stride2_from_l1", ceilings["ldg16_stride2_from_l1"]))}
    first = abs(inner / K - 1.0) < 1e-9          # one descent step per prox call: f is g itself in both passes
    # the trial pass also writes its volume (the result, when the step is accepted and last): + 4 bytes per voxel
    tv_bytes = {"tv_grad": 8.0 if first else 12.0, "tv_trial": 12.0 if first else 16.0, "tv_update": 12.0}
    coop_prox = not per["tv_trial"]["ms_per_launch"] and bool(per["tv_grad"]["ms_per_launch"])
    if coop_prox:
        # the whole prox call is ONE cooperative kernel (timed in the tv_grad slot): per call, a gradient pass of 8 B/voxel
        # (f is g: read g, write d) or 12 (later steps), trial passes of 12 (read g, d; write the candidate) or 16, and an
        # update pass of 12 for every descent step but the last
        i_, t_ = inner / K, trials / K
        tv_bytes = {"tv_grad": 8.0 + 12.0 * max(i_ - 1.0, 0.0) + 12.0 * t_ + 12.0 * max(i_ - 1.0, 0.0)}
    kern = {}
    for name in ("forward", "back"):
        if per[name]["ms_per_launch"]:
            t = per[name]["ms_per_launch"] / 1e3
            kern[name] = {"bound": "l1-gather", "gups": S / t / 1e9, "achieved": 4.0 * S / t / 1e9, "peak": l1_peak_gbs,
                          "unit": "GB/s", "frac": 4.0 * S / t / 1e9 / l1_peak_gbs,
                          "peak_source": "analytic: 148 SMs x 128 B/clk x %.0f MHz (DESIGN.md section 7)" % sm_max_mhz,
                          "peak_measured": measured[name][1], "frac_measured": 4.0 * S / t / 1e9 / measured[name][1],
                          "peak_measured_source": "cbct_gather_ceiling: " + measured[name][0]}
    for name, bpv in tv_bytes.items():
        if per[name]["ms_per_launch"]:
            t = per[name]["ms_per_launch"] / 1e3
            kern["tv_prox" if coop_prox else name] = {
                "bound": "hbm", "achieved": bpv * nvox / t / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "frac": bpv * nvox / t / 1e9 / hbm_peak, "bytes_per_voxel": bpv, "peak_source": peak_src}
    if coop_prox:
        per["tv_prox"] = per["tv_grad"]
    if per["transpose"]["ms_per_launch"]:       # the staging copy: reads the volume, writes the padded z-fastest copy
        t = per["transpose"]["ms_per_launch"] / 1e3
        kern["transpose"] = {"bound": "hbm", "achieved": 8.0 * nvox / t / 1e9, "peak": hbm_peak, "unit": "GB/s",
                             "frac": 8.0 * nvox / t / 1e9 / hbm_peak, "bytes_per_voxel": 8.0, "peak_source": peak_src}
    for name in kern:
        if name in counters:                    # the tracked capture is of this workload and of these kernel sources
            kern[name]["ncu"] = counters[name]
    dominant = max((n for n in kern), key=lambda n: per[n]["ms_per_step"])
    roof = dict(kern[dominant])
    # the same kernel against the HBM roofline, for reference: algorithmic HBM bytes per launch
    alg_hbm = {"back": 4.0 * nray + 8.0 * nvox, "forward": 4.0 * nvox * 1.1 + 8.0 * nray}.get(dominant)
    if alg_hbm is not None:
        t = per[dominant]["ms_per_launch"] / 1e3
        roof["hbm"] = {"algorithmic_bytes": alg_hbm, "achieved": alg_hbm / t / 1e9, "peak": hbm_peak, "unit": "GB/s",
                       "frac": alg_hbm / t / 1e9 / hbm_peak, "peak_source": peak_src}
    roof.update({"kernel": dominant, "traffic": counters.get(dominant, {}).get("dram_bytes_per_launch"),
                 "share_of_step": per[dominant]["ms_per_step"] / sum(v["ms_per_step"] for n_, v in per.items() if n_ != "tv_prox")})
    roof.update(counters_meta)
    roof["back_path"] = back_path

    base = cpu_baseline(cfg, y_host)
    jobs = 1 if sharded else world              # sharded: all ranks worked on the same K steps
    line = {
        "metric": METRIC, "value": aggregate_value(K, jobs, ms_total), "unit": UNIT, "n_gpus": world, "steps": K,
        "warmup": args.warmup, "ms_per_step": ms_total / K,
        "separate_calls_ms_per_step": {"mean": float(np.mean(per_step)), "median": float(np.median(per_step)),
                                       "best": float(np.min(per_step))},
        "higher_is_better": True, "scaling": "strong" if sharded else "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"config{k} ({cfg.name}): {g.nx}x{g.ny}x{g.nz} fp32 voxels at {g.hx} mm, {g.n_proj} views "
                               f"of {g.nu}x{g.nv} at {g.du} mm, one finest-level FBS iteration per step after "
                               f"{n_levels - 1} coarser multi-grid levels",
                   "tv_weight": fbs.tv_weight, "step": fbs.step, "levels": n_levels,
                   "iters_per_level": list(fbs.iters_per_level),
                   "l2": "working set (5 volumes + 2 projection stacks = %.0f MiB) exceeds the 126 MB L2; no flush"
                         % ((5 * nvox + 2 * nray) * 4 / 2 ** 20),
                   "parallelism": ("projectors sharded by output ownership over %d GPUs (cbct_fbs_reconstruct_sharded)" % world
                                   if sharded else "independent problem per GPU" if world > 1 else "single GPU")},
        "clocks": clocks,
        "e2e": {"value": aggregate_value(K, jobs, ms_e2e), "unit": UNIT, "h2d_bytes_per_step": 4 * (nray + nvox),
                "d2h_bytes_per_step": 4 * nvox, "ms_per_step": ms_e2e / K},
        "gpu_launches": int(launches),
        "roofline": roof,
        "gather_ceilings_gbs": {k: round(v, 1) for k, v in ceilings.items()},
        "kernels": kern,
        "stage_ms_per_step": {n: round(v["ms_per_step"], 4) for n, v in per.items()},
        "projector_gups": {"samples_per_projection": int(S),
                           "forward": kern.get("forward", {}).get("gups"), "back": kern.get("back", {}).get("gups")},
        "tv_inner_per_step": inner / K, "tv_trials_per_step": trials / K,
        "cpu_baseline": base,
    }
    if recon:
        line["reconstruction"] = recon
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------------------------
# config 5: projector / TV microbenchmark sweep (each operator alone)
# ---------------------------------------------------------------------------------------------

def run_sweep(args):
    """BASELINE.json config 5: P, P^T and TV-prox each alone on n^3 volumes (n in --sweep-sizes, uniform random in
    [0, 0.03)/mm, fixed 256 mm field of view) with --sweep-views projections of 512x384; prints ONE JSON line whose
    "sweep" list holds, per case, milliseconds per call, projector GUPS and fraction of the L1-gather roofline, and the
    TV passes' achieved HBM GB/s.  Inputs smaller than the 126 MB L2 are followed by an L2 flush between calls."""
    import torch
    from paper_1001_0599_b200 import cbct
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(0)
    hbm_peak, sm_max_mhz, peak_src = _peaks()
    l1_peak_gups = 148 * 128 * sm_max_mhz * 1e6 / 4 / 1e9
    flush = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device="cuda")
    sizes = [int(x) for x in args.sweep_sizes.split(",")]
    views = [int(x) for x in args.sweep_views.split(",")]
    out = []

    def timed(fn, reps):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        for _ in range(3):
            fn()
        for e0, e1 in ev:
            flush.zero_()                       # evict the previous call's lines from L2
            e0.record()
            fn()
            e1.record()
        torch.cuda.synchronize()
        t = sorted(e0.elapsed_time(e1) for e0, e1 in ev)
        return t[len(t) // 2]

    for n in sizes:
        for nv in views:
            g = I.sweep_geometry(n, nv)
            with cbct.geometry_create(g) as h:
                # the seeded host generators of SURVEY.md section 8(d): the inputs tests/test_gpu_fullsize.py checks against the oracle
                f = torch.from_numpy(I.uniform_volume(g, I.SEED_BASE + 5, hi=0.03)).cuda()
                q = torch.from_numpy(I.uniform_projections(g, I.SEED_BASE + 6)).cuda()
                p, b = torch.empty_like(q), torch.empty_like(f)
                S = h.count_samples()
                reps = max(3, min(args.steps, 10))
                case = {"n": n, "n_proj": nv, "symmetry": h.symmetry, "samples": int(S)}
                h.set_stage_timing(True)
                for name, fn, stage in (("forward", lambda: h.forward_project(f, p), "forward"),
                                        ("back", lambda: h.back_project(q, b), "back")):
                    ms = timed(fn, reps)
                    h.set_stage_timing(True)    # reset the accumulators, then attribute the kernel itself
                    fn()
                    kms = h.stage_ms()[stage][0]
                    case[name] = {"ms_per_call": ms, "kernel_ms": kms, "gups": S / kms / 1e6,
                                  "frac_of_l1_gather_roofline": S / kms / 1e6 / l1_peak_gups}
                if nv == views[0]:              # TV does not depend on the view count: once per size
                    setup = I.FbsSetup(max_inner=10, rel_tol=0.0, eps_delta=1e-4)
                    ms = timed(lambda: h.tv_prox(f, b, 1e-3, setup), reps)
                    h.set_stage_timing(True)
                    rep = h.tv_prox(f, b, 1e-3, setup)
                    st = h.stage_ms()
                    nvox = f.numel()
                    tv = {"ms_per_call": ms, "inner_iters": rep.inner_iters, "trials": rep.trials}
                    if st["tv_trial"][1]:               # host-sequenced passes: one kernel each
                        for k, bpv in (("tv_grad", 12.0), ("tv_trial", 12.0), ("tv_update", 12.0)):
                            if st[k][1]:
                                t = st[k][0] / st[k][1]
                                tv[k] = {"ms_per_launch": t, "hbm_gbs": bpv * nvox / t / 1e6,
                                         "frac_of_hbm_peak": bpv * nvox / t / 1e6 / hbm_peak}
                    elif st["tv_grad"][1]:              # the cooperative kernel: every pass of the call in one launch
                        i_, t_ = rep.inner_iters, rep.trials
                        # gradient passes 8 B/voxel (first step: f is g) or 12, trial passes >= 12 (16 once f differs from g;
                        # the report does not split them: a lower bound), an update pass of 12 per step but the last
                        bpv = 8.0 + 12.0 * max(i_ - 1, 0) + 12.0 * t_ + 12.0 * max(i_ - 1, 0)
                        t = st["tv_grad"][0] / st["tv_grad"][1]
                        tv["tv_prox_kernel"] = {"ms_per_launch": t, "bytes_per_voxel_lower_bound": bpv,
                                                "hbm_gbs": bpv * nvox / t / 1e6, "frac_of_hbm_peak": bpv * nvox / t / 1e6 / hbm_peak}
                    case["tv_prox"] = tv
                h.set_stage_timing(False)
                out.append(case)
            del f, q, p, b
            torch.cuda.empty_cache()
    print(json.dumps({"metric": "projector_gups_sweep", "unit": "GUPS", "n_gpus": 1, "data": "synthetic", "dtype": "f32",
                      "config": {"workload": "config5: P, P^T, TV-prox each alone; n^3 volume at 256/n mm, 512x384 detector",
                                 "l2": "256 MiB flush buffer written between timed calls"},
                      "peaks": {"l1_gather_gups": l1_peak_gups, "hbm_gbs": hbm_peak, "source": peak_src},
                      "sweep": out}))


# ---------------------------------------------------------------------------------------------
# Table-1-style sweep: quality metrics and time against the number of views
# ---------------------------------------------------------------------------------------------

def run_table1(args):
    """The shape of the paper's Table 1 on the synthetic torso phantom of config 3: for N_theta in --table1-views, the
    full multi-grid reconstruction (config 3's levels and iteration counts) from N_theta equally spaced noisy views,
    the relative error e and the correlation coefficient c against the voxelised phantom (cbct_quality_metrics) and
    the device time.  Prints ONE JSON line."""
    import torch
    from paper_1001_0599_b200 import cbct
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(0)
    k, cfg = workload(args.workload)
    rows = []
    for n_theta in [int(x) for x in args.table1_views.split(",")]:
        c = I.Config(cfg.name, cfg.geom.replace(n_proj=n_theta, angles=None), cfg.fbs, cfg.ellipsoids, cfg.photons, cfg.seed)
        g = c.geom
        y = torch.from_numpy(I.make_projections(c)).cuda()
        truth = torch.from_numpy(I.paint(c.ellipsoids, g)).cuda()
        with cbct.geometry_create(g, max_levels=len(c.fbs.iters_per_level)) as h:
            f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
            h.fbs_reconstruct(y, f, c.fbs, objective=False)          # warm-up (step bounds are cached in the handle)
            f.zero_()
            rep = h.fbs_reconstruct(y, f, c.fbs, objective=False)
            e, cc = h.quality_metrics(f, truth)
            rows.append({"n_theta": n_theta, "symmetry": h.symmetry, "rel_error_e": e, "correlation_c": cc,
                         "recon_seconds": rep.ms_total / 1e3, "iterations": rep.n_iters_total})
    print(json.dumps({"metric": "table1_quality_vs_views", "n_gpus": 1, "data": "synthetic", "dtype": "f32",
                      "config": {"workload": f"config{k} geometry and phantom, N_theta equally spaced views, "
                                             f"{len(cfg.fbs.iters_per_level)} levels x {list(cfg.fbs.iters_per_level)} iterations",
                                 "tv_weight": cfg.fbs.tv_weight, "step": cfg.fbs.step},
                      "paper_table1": "e = 28.63 / 15.96 / 11.38 / 7.10 %, c = 0.9386 / 0.9813 / 0.9906 / 0.9963, "
                                      "t = 38.7 / 51.2 / 77.8 / 130.3 s for N_theta = 5 / 10 / 20 / 40 on the NCAT phantom, "
                                      "Tesla C1060 (PAPER.md:L255): context, other phantom and hardware",
                      "rows": rows}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config3", choices=["config1", "config2", "config3", "config4"])
    ap.add_argument("--sharded", action="store_true",
                    help="N ranks reconstruct ONE problem, projectors sharded by output ownership (strong scaling); "
                         "default under torchrun: N independent problems (weak scaling)")
    ap.add_argument("--no-recon", action="store_true", help="skip the whole-reconstruction timing")
    ap.add_argument("--no-extra", action="store_true", help="skip the TV-weight scan / field-of-view error beside the headline")
    ap.add_argument("--sweep", action="store_true", help="config 5: operator microbenchmarks instead of the FBS step")
    ap.add_argument("--sweep-sizes", default="64,128,256,512")
    ap.add_argument("--sweep-views", default="1,40,360")
    ap.add_argument("--table1", action="store_true", help="quality metrics and time against the number of views")
    ap.add_argument("--table1-views", default="5,10,20,40")
    args = ap.parse_args()
    if args.sweep:
        return run_sweep(args)
    if args.table1:
        return run_table1(args)
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: note: fewer than 3 warm-up steps", file=sys.stderr)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
