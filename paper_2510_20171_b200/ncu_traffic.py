"""Writes one row of profiles/traffic.csv (DRAM bytes per launch, which bench.py reports as `roofline.traffic`) from
the raw page of an `ncu --set full` capture:

    ncu -i <capture>.ncu-rep --page raw --csv > raw.csv
    python -m paper_2510_20171_b200.ncu_traffic raw.csv segment_copy_kernel cfg3_dispatch "<where the capture came from>"

The raw page has one header row (metric names), one unit row and one row per profiled launch; the LAST launch whose
kernel name contains <kernel> is used.  Measurement tooling only: nothing on the data path imports this module."""
from __future__ import annotations

import csv
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TRAFFIC = os.path.join(ROOT, "profiles", "traffic.csv")
SCALE = {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
FIELDS = ["kernel", "workload", "dram_bytes_read", "dram_bytes_write", "bytes_per_launch", "source"]


def dram_bytes(raw_csv: str, kernel: str):
    """-> (bytes read, bytes written) of the last launch of `kernel` in an ncu raw-page CSV."""
    rows = [r for r in csv.reader(open(raw_csv)) if r]
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    hdr, units, body = rows[start], rows[start + 1], rows[start + 2:]
    k = hdr.index("Kernel Name")
    hits = [r for r in body if kernel in r[k]]
    if not hits:
        raise SystemExit(f"no launch of {kernel!r} in {raw_csv}")
    out = []
    for name in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
        i = hdr.index(name)
        out.append(int(round(float(hits[-1][i].replace(",", "")) * SCALE[units[i]])))
    return out[0], out[1]


def update(path: str, kernel: str, workload: str, rd: int, wr: int, source: str) -> None:
    rows = list(csv.DictReader(open(path))) if os.path.exists(path) else []
    rows = [r for r in rows if not (r["kernel"] == kernel and r["workload"] == workload)]
    rows.append({"kernel": kernel, "workload": workload, "dram_bytes_read": rd, "dram_bytes_write": wr,
                 "bytes_per_launch": rd + wr, "source": source})
    with open(path, "w", newline="") as f:
        w = csv.DictWriter(f, FIELDS, lineterminator="\n")
        w.writeheader()
        w.writerows(rows)


if __name__ == "__main__":
    if len(sys.argv) != 5:
        raise SystemExit(__doc__)
    raw, kernel, workload, source = sys.argv[1:]
    rd, wr = dram_bytes(raw, kernel)
    update(TRAFFIC, kernel, workload, rd, wr, source)
    print(f"{kernel},{workload}: read {rd} + write {wr} = {rd + wr} bytes per launch -> {TRAFFIC}")
