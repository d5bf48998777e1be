"""NEXT-4: the reconstruction sharded by output ownership (include/cbct.h: cbct_fbs_reconstruct_sharded).

* CPU, world_size 2 over gloo: the partition arithmetic every rank evaluates on its own (cbct_shard_range) tiles the
  units exactly, whatever the counts, and the chunks the ranks exchange (residual-stack chunks per base view, slabs of the
  volume with their mirror images) cover every element exactly once.
* GPU (one device): TWO ranks emulated by two host threads, each with its own handle and stream, whose collectives are device
  copies between the two handles' buffers; the volume of either rank must be BIT FOR BIT the single-GPU reconstruction's.
  (Kernels of the two ranks never wait on one another on the device: the hand-over is a host barrier between stream
  synchronisations.)  A real multi-GPU run needs a multi-GPU box; the test of that is below and skips itself.
"""
import os
import socket
import sys
import threading

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1001_0599_b200 import inputs as I  # noqa: E402


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _partition_worker(rank: int, world: int, port: int):
    os.environ.update({"MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    sys.path.insert(0, ROOT)
    from paper_1001_0599_b200 import cbct
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # (units, nz, z-unit slices, mirror symmetric?) -- config 3 (10 base views; 4 z-units of 32 of the lower 128 slices),
    # config 4 (90 base views, list kernel: 2 z-units of 64), odd counts, fewer units than ranks
    for n_base, nz, unit, mirror in ((10, 256, 32, True), (90, 256, 64, True), (7, 19, 32, False), (1, 40, 32, True), (3, 96, 32, False)):
        nzh = nz // 2 if mirror else nz
        n_zu = (nzh + unit - 1) // unit
        mine = torch.tensor(list(cbct.shard_range(n_base, world, rank)) + list(cbct.shard_range(n_zu, world, rank)))
        every = [torch.zeros_like(mine) for _ in range(world)]
        dist.all_gather(every, mine)
        every = [e.tolist() for e in every]
        # base views: contiguous, ordered, balanced
        assert every[0][0] == 0 and every[-1][1] == n_base
        assert all(every[r][1] == every[r + 1][0] for r in range(world - 1))
        sizes = [e[1] - e[0] for e in every]
        assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
        # slabs of the volume: every slice owned exactly once (a z-unit and, with mirror symmetry, its mirror image)
        owner = np.zeros(nz, dtype=int)
        for e in every:
            k_lo, k_hi = e[2] * unit, min(e[3] * unit, nzh)
            if k_hi > k_lo:
                owner[k_lo:k_hi] += 1
                if mirror:
                    owner[nz - k_hi:nz - k_lo] += 1
        assert (owner == 1).all(), (n_base, nz, unit, mirror, owner)
    dist.barrier()
    dist.destroy_process_group()


def test_partition_tiles_views_and_slabs_world2():
    mp.spawn(_partition_worker, args=(2, _free_port()), nprocs=2, join=True)


def test_shard_range_is_balanced_and_rejects_nonsense():
    from paper_1001_0599_b200 import cbct
    for n in (0, 1, 5, 10, 90, 97):
        for world in (1, 2, 3, 8):
            parts = [cbct.shard_range(n, world, r) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
            assert max(hi - lo for lo, hi in parts) - min(hi - lo for lo, hi in parts) <= 1
    with pytest.raises(cbct.CbctError):
        cbct.shard_range(4, 2, 2)
    with pytest.raises(cbct.CbctError):
        cbct.shard_range(4, 0, 0)


# ---------------------------------------------------------------------------------------------------------------------
# GPU: two emulated ranks on one device
# ---------------------------------------------------------------------------------------------------------------------

class _ThreadFabric:
    """The collectives of `world` emulated ranks living in one process: device copies between the ranks' buffers, handed
    over through host barriers placed between stream synchronisations."""

    def __init__(self, world):
        self.world = world
        self.barrier = threading.Barrier(world)
        self.slot = [None] * world

    def comm(self, cbct, rank):
        def post(t):
            torch.cuda.current_stream().synchronize()          # my part of the buffer is complete
            self.slot[rank] = t
            self.barrier.wait()

        def broadcast(t, root):
            post(t)
            if rank != root:
                t.copy_(self.slot[root])
                torch.cuda.current_stream().synchronize()
            self.barrier.wait()

        def allreduce_sum(t):
            post(t)
            total = self.slot[0].clone()
            for r in range(1, self.world):
                total += self.slot[r]                            # rank order; every slot but one holds 0: exact
            torch.cuda.current_stream().synchronize()
            self.barrier.wait()                                  # everyone has read everyone's buffer
            t.copy_(total)
            torch.cuda.current_stream().synchronize()
            self.barrier.wait()

        return cbct.Comm(rank, self.world, broadcast, allreduce_sum)


@pytest.mark.gpu
@pytest.mark.parametrize("world,case", [(2, "tma"), (3, "tma"), (2, "list")])
def test_sharded_reconstruction_equals_single_gpu_bitwise(world, case):
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_1001_0599_b200 import cbct
    if case == "tma":       # quarter-turn + mirror symmetric, voxel shadow ~1.9 columns: the TMA back-projector, 3 z-units
        g = I.Geometry(nx=48, ny=48, nz=192, hx=2.0, hy=2.0, hz=1.0, nu=64, nv=96, du=1.6, dv=0.8, sad=1000.0, sdd=1500.0,
                       n_proj=20)
    else:                   # a 200-degree arc: no quarter-turn symmetry, the list kernel, 40 base views
        g = I.Geometry(nx=48, ny=48, nz=160, hx=2.0, hy=2.0, hz=1.0, nu=64, nv=80, du=2.4, dv=1.2, sad=1000.0, sdd=1500.0,
                       n_proj=40, angles=np.deg2rad(200.0) * np.arange(40) / 40)
    ell = [I.Ellipsoid((0.0, 0.0, 0.0), (40.0, 34.0, 70.0), 0.0, 0.02)] + \
        I.random_ellipsoids(np.random.default_rng(141), 6, (48.0, 48.0, 80.0), axes_range=(4.0, 14.0))
    y = torch.from_numpy(I.poisson_log(I.analytic_projections(ell, g), 1e5, 142).astype(np.float32)).cuda()
    setup = I.FbsSetup(iters_per_level=(3, 3), tv_weight=30.0)
    with cbct.geometry_create(g, max_levels=2) as h:
        assert h.back_path(0) == case
        n_base, n_zu, unit = h.shard_units(0)
        assert n_zu >= 2 and n_base >= world
        f1 = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        rep1 = h.fbs_reconstruct(y, f1, setup)
        want = f1.cpu().numpy()
    fabric = _ThreadFabric(world)
    outs, reps, errs = [None] * world, [None] * world, []

    def rank_main(rank):
        try:
            torch.cuda.set_device(0)
            stream = torch.cuda.Stream()
            with torch.cuda.stream(stream), cbct.geometry_create(g, max_levels=2) as h:
                f = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
                reps[rank] = h.fbs_reconstruct_sharded(fabric.comm(cbct, rank), y, f, setup, stream=stream)
                outs[rank] = f.cpu().numpy()
        except Exception as e:          # a dead rank would leave the others at a barrier
            errs.append(e)
            fabric.barrier.abort()

    threads = [threading.Thread(target=rank_main, args=(r,)) for r in range(world)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=600)
    assert not errs, errs
    for r in range(world):
        assert outs[r].tobytes() == want.tobytes(), (r, float(np.abs(outs[r] - want).max()))
        assert np.array_equal(reps[r].objective, rep1.objective)         # the E2 sums are formed in the single-GPU order
        assert (reps[r].inner_total, reps[r].trials_total) == (rep1.inner_total, rep1.trials_total)


@pytest.mark.gpu
def test_sharded_reconstruction_on_two_real_gpus():
    """The same comparison over NCCL on two devices (torch.distributed, one process per GPU)."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    mp.spawn(_nccl_worker, args=(2, _free_port()), nprocs=2, join=True)


def _nccl_worker(rank, world, port):
    os.environ.update({"MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    sys.path.insert(0, ROOT)
    from paper_1001_0599_b200 import cbct
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    g = I.Geometry(nx=48, ny=48, nz=192, hx=2.0, hy=2.0, hz=1.0, nu=64, nv=96, du=1.6, dv=0.8, sad=1000.0, sdd=1500.0, n_proj=20)
    ell = [I.Ellipsoid((0.0, 0.0, 0.0), (40.0, 34.0, 70.0), 0.0, 0.02)]
    y = torch.from_numpy(I.poisson_log(I.analytic_projections(ell, g), 1e5, 142).astype(np.float32)).cuda()
    setup = I.FbsSetup(iters_per_level=(3, 3), tv_weight=30.0)
    with cbct.geometry_create(g, max_levels=2) as h:
        f1 = torch.zeros(g.vol_shape, device="cuda", dtype=torch.float32)
        h.fbs_reconstruct(y, f1, setup)
        f = torch.zeros_like(f1)
        h.fbs_reconstruct_sharded(cbct.torch_distributed_comm(), y, f, setup)
        assert torch.equal(f, f1)
    dist.destroy_process_group()
