"""Records the DRAM traffic of a kernel from an `ncu --set full` capture in profiles/traffic.json.

    ncu -i gpurun_out/<capture>.ncu-rep --page raw --csv --print-units base \\
        | python -m paper_2509_06525_b200.ncu_traffic <quantity> <workload name> <kernel substring> <source .md>

<quantity> is bench.py's key ("dos", "dos-sp", "dos-spd", "dos-spd-bond", "vac", ...).  The value stored is
the mean over the matching launches of dram__bytes_read.sum + dram__bytes_write.sum, per launch, which
bench.py prints as roofline.traffic.  No arithmetic of the method lives here.
"""
from __future__ import annotations

import csv
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PATH = os.path.join(ROOT, "profiles", "traffic.json")


def dram_bytes_per_launch(rows, kernel_substring: str):
    header = rows[0]
    name_col = header.index("Kernel Name")
    rd, wr = header.index("dram__bytes_read.sum"), header.index("dram__bytes_write.sum")
    units = rows[1]
    for col in (rd, wr):
        if units[col] not in ("byte", "bytes", ""):
            raise SystemExit(f"expected bytes (use --print-units base), got unit {units[col]!r}")
    vals = [float(r[rd].replace(",", "")) + float(r[wr].replace(",", ""))
            for r in rows[2:] if len(r) > max(rd, wr) and kernel_substring in r[name_col]]
    vals = [v for v in vals if v == v]          # a launch the capture cut short reads nan
    if not vals:
        raise SystemExit(f"no launch of a kernel matching {kernel_substring!r} in the capture")
    return sum(vals) / len(vals), len(vals)


def main(argv):
    if len(argv) != 5:
        raise SystemExit(__doc__)
    quantity, workload, kernel, source = argv[1:]
    rows = [r for r in csv.reader(sys.stdin) if r]
    while rows and "Kernel Name" not in rows[0]:      # ncu prints "==PROF==" lines before the table
        rows.pop(0)
    value, count = dram_bytes_per_launch(rows, kernel)
    data = {}
    if os.path.exists(PATH):
        with open(PATH) as f:
            data = json.load(f)
    data.setdefault(quantity, {})[workload] = {"dram_bytes_per_launch": value, "kernel": kernel,
                                               "launches": count, "source": source}
    with open(PATH, "w") as f:
        json.dump(data, f, indent=2)
        f.write("\n")
    print(f"{quantity} / {workload}: {value / 1e9:.4f} GB per launch over {count} launches of {kernel}")


if __name__ == "__main__":
    main(sys.argv)
