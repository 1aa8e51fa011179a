"""Turn an Nsight Compute report of the library's kernels into the small JSON file bench.py reads.

    python -m paper_1506_08481_b200.profile_counters gpurun_out/prof.ncu-rep "<capture command>" > profiles/r02_counters.json

Reads the report with ``ncu -i <report> --page raw --csv`` (no GPU needed) and keeps, per kernel (first captured
launch of each name, template arguments stripped), the counters the roofline object of bench.py quotes: DRAM bytes
read and written, duration under the profiler, FP64 pipe activity, executed FP64 warp instructions, registers,
grid and block size.  Nothing here touches the device or the product path.
"""
from __future__ import annotations

import csv
import io
import json
import re
import subprocess
import sys

_KEEP = {
    "gpu__time_duration.sum": "duration",
    "dram__bytes_read.sum": "dram_bytes_read",
    "dram__bytes_write.sum": "dram_bytes_write",
    "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active": "fp64_pipe_active_pct",
    "smsp__inst_executed_pipe_fp64.sum": "fp64_warp_instructions",
    "smsp__inst_executed.sum": "warp_instructions",
    "smsp__thread_inst_executed_per_inst_executed.ratio": "active_threads_per_instruction",
    "sm__warps_active.avg.pct_of_peak_sustained_active": "warps_active_pct",
    "launch__registers_per_thread": "registers_per_thread",
    "launch__grid_size": "grid_size",
    "launch__block_size": "block_size",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum": "shared_wavefronts",
}
_SCALE = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "ms": 1e-3, "us": 1e-6, "ns": 1e-9, "s": 1.0, "second": 1.0,
          "msecond": 1e-3, "usecond": 1e-6, "nsecond": 1e-9}


def counters(report: str) -> dict:
    out = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    hdr, units = rows[0], rows[1]
    iname = hdr.index("Kernel Name")
    kernels = {}
    for r in rows[2:]:
        name = re.sub(r"^void\s+", "", r[iname])
        name = re.split(r"[<(]", name)[0].strip()
        if name in kernels:
            name = f"{name}#{sum(1 for k in kernels if k.split('#')[0] == name) + 1}"
        entry = {"kernel": r[iname].split("(")[0]}
        for metric, key in _KEEP.items():
            if metric in hdr:
                i = hdr.index(metric)
                try:
                    entry[key] = float(r[i].replace(",", "")) * _SCALE.get(units[i], 1.0)
                except ValueError:
                    entry[key] = None
        kernels[name] = entry
    return kernels


def main(argv):
    if len(argv) < 2:
        print(__doc__, file=sys.stderr)
        return 2
    doc = {"report": argv[1], "command": argv[2] if len(argv) > 2 else None,
           "units": "bytes, seconds, percent, counts; per launch, under the profiler (cold caches, serialised)",
           "kernels": counters(argv[1])}
    json.dump(doc, sys.stdout, indent=1)
    print()
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv))
