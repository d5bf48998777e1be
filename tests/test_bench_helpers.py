"""Host-side helpers of the measurement: the field-of-view mask of bench.py and the ncu counters record."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1001_0599_b200 import inputs as I  # noqa: E402
from paper_1001_0599_b200 import ncu_counters  # noqa: E402


def test_fov_mask_is_the_cone_seen_by_every_view():
    import bench
    g = I.config(1).geom                       # 32^3 at 2 mm, 48x48 detector at 1.6 mm: 76.8 mm covers ~51 mm at the isocentre
    m = bench.fov_mask(g)
    assert m.shape == g.vol_shape and m.dtype == bool
    c = g.nz // 2
    assert m[c, g.ny // 2, g.nx // 2] and m[c - 1, g.ny // 2 - 1, g.nx // 2 - 1]     # around the isocentre: seen
    assert not m[0].any() and not m[-1].any()                                           # top / bottom slices: outside the cone
    assert not m[c, 0, 0]                                                                # in-plane corner: outside the fan
    assert np.array_equal(m, m[::-1])                                                    # mirror symmetric in z
    assert np.array_equal(m[c], m[c].T)                                                  # 8 equally spaced views: quarter-turn symmetric
    # the voxel column next to the axis is seen while |z| <= v_max * (depth of the view that sees least of it) / sdd
    zc = (np.arange(g.nz) - 0.5 * (g.nz - 1)) * g.hz
    x1 = 0.5 * g.hx                                                 # even nx: the four columns around the axis are at (+-h/2, +-h/2)
    depth_min = g.sad - np.hypot(x1, x1)                            # 8 views at multiples of 45 degrees: one looks along the diagonal
    limit = 0.5 * g.nv * g.dv * depth_min / g.sdd
    col = m[:, g.ny // 2, g.nx // 2]
    clear = np.abs(np.abs(zc) - limit) > 0.1                       # no slice centre sits on the limit
    assert clear.all() and np.array_equal(col, np.abs(zc) <= limit)


def test_ncu_counters_record_parses_a_raw_export(tmp_path):
    raw = tmp_path / "raw.csv"
    hdr = ["ID", "Kernel Name", "Grid Size", "Block Size", "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum",
           "l1tex__t_sector_hit_rate.pct", "launch__registers_per_thread"]
    units = ["", "", "", "", "us", "Mbyte", "Mbyte", "%", "register/thread"]
    rows = [["0", "void <unnamed>::back_tma_kernel<4, 4, 1, 3, 2, 2>(BtMaps, LevelParams)", "(32, 32, 4)", "(544, 1, 1)", "889.1", "99.5", "44.3", "64.5", "56"],
            ["1", "void forward_kernel<4, 2, 1>(LevelParams, const void *)", "(64, 10, 6)", "(32, 8, 1)", "766.0", "99.3", "21.2", "68.2", "76"],
            ["2", "void forward_kernel<4, 2, 1>(LevelParams, const void *)", "(64, 10, 6)", "(32, 8, 1)", "1.0", "1.0", "1.0", "1.0", "76"],
            ["3", "stage_volume_packed_vec_kernel(const float *, float4 *, int, int, int, int, int)", "(4, 5, 256)", "(256, 1, 1)", "23.3", "67.1", "24.6", "1.0", "28"],
            ["4", "void tv_prox_coop_kernel<1>(TvCoop)", "(576, 1, 1)", "(32, 4, 1)", "111.0", "222.2", "85.5", "2.0", "128"]]
    raw.write_text("\n".join(",".join('"%s"' % c for c in r) for r in [hdr, units] + rows))
    k = ncu_counters.parse(str(raw))
    assert set(k) == {"back", "forward", "transpose", "tv_prox"}
    assert k["transpose"]["registers"] == 28 and k["tv_prox"]["ncu_duration_us"] == 111.0
    assert k["back"]["dram_bytes_per_launch"] == 99.5e6 + 44.3e6 and k["back"]["registers"] == 56
    assert k["forward"]["ncu_duration_us"] == 766.0            # the FIRST launch of a kernel
    h = ncu_counters.kernel_sources_sha256()
    assert len(h) == 64 and h == ncu_counters.kernel_sources_sha256()


def test_tracked_counters_record_is_well_formed():
    p = os.path.join(ROOT, "profiles", "r02_counters.json")
    rec = json.load(open(p))
    assert len(rec["kernel_sources_sha256"]) == 64 and rec["ncu_command"].startswith("ncu ")
    assert {"forward", "back", "tv_prox", "transpose"} <= set(rec["kernels"])
    for k in rec["kernels"].values():
        assert k["dram_bytes_per_launch"] > 0
