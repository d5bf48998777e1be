"""Turn an `ncu --page raw --csv` export of a bench.py capture into the counters record bench.py quotes.

    ncu -i gpurun_out/prof.ncu-rep --page raw --csv > raw.csv
    python -m paper_1001_0599_b200.ncu_counters raw.csv "<the ncu command line>" > profiles/r02_counters.json

The record holds, per kernel of the FBS step, the memory-path evidence BASELINE.json's north_star asks for (DRAM bytes
per launch, L1 / L2 hit rates, l1tex / lts / issue utilisation, registers, occupancy) and is stamped with a hash of the
kernel sources it was captured from: bench.py prints these counters only while the sources still hash to the same value.
"""
from __future__ import annotations

import csv
import hashlib
import json
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")

# kernel-name prefix -> bench.py's stage name
STAGES = {"forward_kernel": "forward", "forward_fold_kernel": "forward", "stage_volume_fold_kernel": "transpose",
          "back_tma_kernel": "back", "back_list_kernel": "back", "back_kernel": "back",
          "tv_grad_kernel": "tv_grad", "tv_energy_kernel": "tv_trial", "tv_update_kernel": "tv_update",
          "stage_volume_packed_kernel": "transpose", "stage_volume_packed_vec_kernel": "transpose",
          "stage_volume_kernel": "transpose", "tv_prox_coop_kernel": "tv_prox"}
METRICS = {
    "gpu__time_duration.sum": "ncu_duration_us",
    "dram__bytes_read.sum": "dram_read_bytes",
    "dram__bytes_write.sum": "dram_write_bytes",
    "lts__t_sector_hit_rate.pct": "l2_hit_pct",
    "l1tex__t_sector_hit_rate.pct": "l1_hit_pct",
    "l1tex__throughput.avg.pct_of_peak_sustained_elapsed": "l1tex_throughput_pct",
    "lts__throughput.avg.pct_of_peak_sustained_elapsed": "lts_throughput_pct",
    "dram__throughput.avg.pct_of_peak_sustained_elapsed": "dram_throughput_pct",
    "smsp__issue_active.avg.pct_of_peak_sustained_active": "issue_active_pct",
    "sm__warps_active.avg.pct_of_peak_sustained_active": "occupancy_pct",
    "launch__registers_per_thread": "registers",
    "smsp__inst_executed.sum": "warp_instructions",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum": "shared_wavefronts",
    "l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum": "l1_global_load_sectors",
    "l1tex__data_pipe_lsu_wavefronts.sum": "l1_data_pipe_wavefronts",
    "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed": "l1_data_pipe_pct",
    "l1tex__t_requests_pipe_lsu_mem_global_op_ld.sum": "l1_global_load_requests",
}
UNIT_SCALE = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "ms": 1e3, "us": 1.0, "ns": 1e-3, "s": 1e6, "second": 1e6,
              "msecond": 1e3, "usecond": 1.0, "nsecond": 1e-3}


def kernel_sources_sha256() -> str:
    """Hash of every file under csrc/ and of include/cbct.h (names and contents, sorted)."""
    h = hashlib.sha256()
    files = sorted(os.listdir(CSRC))
    for name in files:
        if name.endswith((".cu", ".cuh", ".h")):
            h.update(name.encode())
            h.update(open(os.path.join(CSRC, name), "rb").read())
    h.update(open(os.path.join(HERE, "..", "include", "cbct.h"), "rb").read())
    return h.hexdigest()


def parse(raw_csv: str) -> dict:
    rows = list(csv.reader(open(raw_csv)))
    hdr, units, data = rows[0], rows[1], rows[2:]
    ix = {h: i for i, h in enumerate(hdr)}
    out = {}
    for r in data:
        name = r[ix["Kernel Name"]]
        stage = next((st for k, st in sorted(STAGES.items(), key=lambda kv: -len(kv[0])) if k in name), None)
        if stage is None or stage in out:
            continue                                    # first launch of each kernel
        rec = {"kernel": name.split("(")[0].strip(), "grid": r[ix["Grid Size"]], "block": r[ix["Block Size"]]}
        for m, key in METRICS.items():
            if m not in ix:
                continue
            try:
                v = float(r[ix[m]].replace(",", ""))
            except ValueError:
                continue
            rec[key] = v * UNIT_SCALE.get(units[ix[m]], 1.0)
        if "dram_read_bytes" in rec and "dram_write_bytes" in rec:
            rec["dram_bytes_per_launch"] = rec["dram_read_bytes"] + rec["dram_write_bytes"]
        out[stage] = rec
    return out


def main(argv):
    if len(argv) < 2:
        sys.exit(__doc__)
    try:
        commit = subprocess.run(["git", "rev-parse", "HEAD"], cwd=HERE, capture_output=True, text=True).stdout.strip()
    except OSError:
        commit = ""
    rec = {"counters_commit": commit, "kernel_sources_sha256": kernel_sources_sha256(),
           "ncu_command": argv[2] if len(argv) > 2 else "", "note": "one launch per kernel, cold-cache and serialised under ncu: "
           "evidence for the memory path, not a timing", "kernels": parse(argv[1])}
    print(json.dumps(rec, indent=1))


if __name__ == "__main__":
    main(sys.argv)
