"""Post-process an `ncu --set full` capture into profiles/dram_traffic.csv (read by bench.py's roofline).

    ncu -i capture.ncu-rep --page raw --csv > capture.raw.csv
    python -m paper_2506_20513_b200.ncu_traffic --config 4 --part adj --raw-csv capture.raw.csv \
        --kernel adj_kernel --cell-steps 148484800 --source profiles/r02_ncu_full_adj_config4.csv

`--part` is one of fwd (first forward sweep), recompute (forward-type sweep that writes every Ez plane
of a checkpoint segment) or adj; `--cell-steps` is what ONE captured launch advances: shots in the
launch x nz x nx x fused steps.  The entry is keyed by the config and by a hash of csrc/ (the GPU box has
no .git), so bench.py can tell when the kernels have changed since the capture (`traffic_stale`).
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import os
import re
import statistics

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
TABLE = os.path.join(_ROOT, "profiles", "dram_traffic.csv")
FIELDS = ["config", "kernel_source_sha", "part", "dram_bytes_per_cell_step", "launches", "grid",
          "cell_steps_per_launch", "dram_read_bytes", "dram_write_bytes", "duration_us_under_ncu", "source"]
_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
          "ns": 1e-9, "us": 1e-6, "ms": 1e-3, "s": 1.0, "usecond": 1e-6, "msecond": 1e-3, "nsecond": 1e-9,
          "second": 1.0}


def kernel_source_sha() -> str:
    h = hashlib.sha256()
    d = os.path.join(_HERE, "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith(".cuh"):            # the device code (kernels); host-only edits do not count
            with open(os.path.join(d, f), "rb") as fh:
                h.update(f.encode()); h.update(fh.read())
    return h.hexdigest()[:16]


def read_table():
    """Rows of profiles/dram_traffic.csv (oldest first), [] if the table does not exist."""
    if not os.path.exists(TABLE):
        return []
    with open(TABLE, newline="") as f:
        return list(csv.DictReader(f))


def read_raw(path: str, kernel_regex: str, grid: str | None = None):
    """-> list of dict(read, write, seconds) per captured launch whose kernel name matches."""
    with open(path, newline="") as f:
        rows = [r for r in csv.reader(f) if r]
    start = next(i for i, r in enumerate(rows) if r[0] == "ID")
    head, units, data = rows[start], rows[start + 1], rows[start + 2:]
    col = {n: i for i, n in enumerate(head)}

    def val(r, name):
        i = col[name]
        return float(r[i].replace(",", "")) * _SCALE[units[i]]

    out = []
    for r in data:
        if len(r) < len(head) or not re.search(kernel_regex, r[col["Kernel Name"]]):
            continue
        if grid is not None and r[col["Grid Size"]].replace(" ", "") != grid.replace(" ", ""):
            continue
        out.append({"read": val(r, "dram__bytes_read.sum"), "write": val(r, "dram__bytes_write.sum"),
                    "seconds": val(r, "gpu__time_duration.sum"), "grid": r[col["Grid Size"]],
                    "kernel": r[col["Kernel Name"]]})
    return out


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--part", choices=["fwd", "recompute", "adj"], required=True)
    ap.add_argument("--raw-csv", required=True)
    ap.add_argument("--kernel", required=True, help="regex on the kernel name")
    ap.add_argument("--cell-steps", type=float, required=True, help="cell-steps one captured launch advances")
    ap.add_argument("--source", required=True, help="the tracked profiles/ file the capture is summarised in")
    ap.add_argument("--sha", default=None, help="csrc hash of the captured build (default: the tree's)")
    ap.add_argument("--grid", default=None, help='only launches with this grid, e.g. "(18, 38, 1)"')
    a = ap.parse_args()
    launches = read_raw(a.raw_csv, a.kernel, a.grid)
    if not launches:
        raise SystemExit("no launch of that kernel in the capture")
    per = statistics.mean((l["read"] + l["write"]) for l in launches) / a.cell_steps
    sha = a.sha or kernel_source_sha()
    row = {"config": str(a.config), "kernel_source_sha": sha, "part": a.part,
           "dram_bytes_per_cell_step": f"{per:.3f}", "launches": str(len(launches)), "grid": launches[0]["grid"],
           "cell_steps_per_launch": f"{a.cell_steps:.0f}",
           "dram_read_bytes": f"{statistics.mean(l['read'] for l in launches):.0f}",
           "dram_write_bytes": f"{statistics.mean(l['write'] for l in launches):.0f}",
           "duration_us_under_ncu": f"{statistics.mean(l['seconds'] for l in launches) * 1e6:.2f}",
           "source": a.source}
    rows = read_table()
    rows = [r for r in rows if (r["config"], r["kernel_source_sha"], r["part"]) != (row["config"], sha, a.part)]
    rows.append(row)
    with open(TABLE, "w", newline="") as f:
        w = csv.DictWriter(f, fieldnames=FIELDS)
        w.writeheader()
        w.writerows(rows)
    print(f"config {a.config} {a.part}: {per:.2f} B per cell-step over {len(launches)} launch(es) -> {TABLE}")


if __name__ == "__main__":
    main()
