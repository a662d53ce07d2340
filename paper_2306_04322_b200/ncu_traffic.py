"""Writes profiles/ncu_traffic.json entries from an ncu capture -- the only way those figures get there.

    ncu --set full --clock-control none -k regex:'row_kernel|col2d_kernel|col_kernel' -s <skip> -c <n> -o cap \\
        python bench.py --steps 20 --warmup 5 --no-cpu-baseline --no-cufft --no-small-grids --workload W --also
    ncu -i cap.ncu-rep --page raw --csv > cap.csv
    python -m paper_2306_04322_b200.ncu_traffic --workload W --csv cap.csv --capture "<the ncu command above>"

For every step kernel found in the CSV the entry  traffic[W][kernel] = {dram_bytes_per_launch, launches, source_hash, capture}
is replaced: dram__bytes_read.sum + dram__bytes_write.sum averaged over the captured launches of that kernel, and the hash of
the files that kernel is compiled from AS THEY ARE NOW (run this from the tree the capture was taken from). bench.py quotes a
figure as `roofline.traffic` only while that hash still matches, and prints null otherwise; nobody edits the hash by hand.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import json
import os
import re

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
JSON_PATH = os.path.join(os.path.dirname(HERE), "profiles", "ncu_traffic.json")

# the files each step kernel is compiled from: its .cu and every header it includes (directly or not)
KERNEL_SOURCES = {
    "row_c2r_nonlinear_r2c": ["row_kernels.cu", "pf_kernels.cuh", "fft_core.cuh"],
    "col_y_fft_update_ifft": ["col2d_kernels.cu", "pf_kernels.cuh", "col_buf.cuh", "fft_core.cuh"],
    "col_y_fwd": ["col_kernels.cu", "pf_kernels.cuh", "col_buf.cuh", "wfft.cuh", "fft_core.cuh"],
    "col_z_fft_update_ifft": ["col_kernels.cu", "pf_kernels.cuh", "col_buf.cuh", "wfft.cuh", "fft_core.cuh"],
    "col_y_inv": ["col_kernels.cu", "pf_kernels.cuh", "col_buf.cuh", "wfft.cuh", "fft_core.cuh"],
}
_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
_COL_MODE = {1: "col_y_fwd", 2: "col_y_inv", 3: "col_z_fft_update_ifft"}     # ColMode of pf_kernels.cuh


def source_hash(kernel=None) -> str:
    """Hash of the sources of one step kernel (None: of every kernel file and header)."""
    if kernel is None:
        files = [f for f in sorted(os.listdir(CSRC)) if f.endswith(".cuh") or f.endswith("_kernels.cu")]
    else:
        files = KERNEL_SOURCES[kernel]
    h = hashlib.sha256()
    for f in files:
        with open(os.path.join(CSRC, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def step_kernel_of(function_name: str):
    """Maps a CUDA function name as ncu prints it to the step-kernel name pf_fs_kernel_name reports (None: not a step kernel)."""
    if "row_kernel<" in function_name:
        m = re.search(r"row_kernel<\w+, \d+, \d+, (\d+)", function_name)
        return "row_c2r_nonlinear_r2c" if m and int(m.group(1)) == 1 else None           # MODE 1 = ROW_STEP
    if "col2d_kernel<" in function_name:
        return "col_y_fft_update_ifft"
    m = re.search(r"col_kernel<\w+, \d+, \d+, \d+, (\d+)>", function_name)
    if m:
        return _COL_MODE.get(int(m.group(1)))
    return None


def parse(csv_path: str):
    """{step kernel: [dram bytes of each captured launch]} from `ncu --page raw --csv` (wide) or `ncu --csv` (long) output."""
    with open(csv_path, newline="") as fh:
        rows = [r for r in csv.reader(fh) if r]
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    head, body = rows[start], rows[start + 1:]
    per = {}
    if "Metric Name" in head:                                   # long format: one row per (launch, metric)
        ki, ii, mi, ui, vi = (head.index(k) for k in ("Kernel Name", "ID", "Metric Name", "Metric Unit", "Metric Value"))
        acc = {}
        for r in body:
            if r[mi] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                acc.setdefault((r[ii], r[ki]), 0.0)
                acc[(r[ii], r[ki])] += float(r[vi].replace(",", "")) * _UNIT[r[ui]]
        for (_, fn), v in acc.items():
            k = step_kernel_of(fn)
            if k:
                per.setdefault(k, []).append(v)
        return per
    ki, ri, wi = head.index("Kernel Name"), head.index("dram__bytes_read.sum"), head.index("dram__bytes_write.sum")
    gi = head.index("Grid Size") if "Grid Size" in head else None
    units = body[0]                                             # wide format: the second row holds the units
    grids = {}
    for r in body[1:]:
        k = step_kernel_of(r[ki])
        if k:
            g = tuple(int(v) for v in re.findall(r"\d+", r[gi])) if gi is not None else ()
            grids.setdefault(k, {}).setdefault(g, []).append(
                float(r[ri].replace(",", "")) * _UNIT[units[ri]] + float(r[wi].replace(",", "")) * _UNIT[units[wi]])
    # col2d_kernel also serves the one-off pass that fills the carried spectrum after pf_set_fields, with a smaller grid:
    # a step launch is the one with the most CTAs
    for k, by_grid in grids.items():
        per[k] = by_grid[max(by_grid, key=lambda g: (g[0] * (g[1] if len(g) > 1 else 1) * (g[2] if len(g) > 2 else 1)) if g else 0)]
    return per


def update(workload: str, csv_path: str, capture: str, json_path: str = JSON_PATH):
    try:
        with open(json_path) as fh:
            doc = json.load(fh)
    except FileNotFoundError:
        doc = {}
    doc = {"format": "traffic[workload][kernel] = {dram_bytes_per_launch, launches, source_hash, capture}; written by "
                     "python -m paper_2306_04322_b200.ncu_traffic, quoted by bench.py while source_hash matches",
           "traffic": {w: {k: e for k, e in ks.items() if isinstance(e, dict)} for w, ks in doc.get("traffic", {}).items()}}
    per = parse(csv_path)
    for k, vals in per.items():
        doc["traffic"].setdefault(workload, {})[k] = {"dram_bytes_per_launch": sum(vals) / len(vals), "launches": len(vals),
                                                      "source_hash": source_hash(k), "capture": capture}
    with open(json_path, "w") as fh:
        json.dump(doc, fh, indent=1)
        fh.write("\n")
    return per


if __name__ == "__main__":
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--workload", required=True)
    ap.add_argument("--csv", required=True)
    ap.add_argument("--capture", required=True, help="the full ncu command the CSV came from")
    ap.add_argument("--json", default=JSON_PATH)
    a = ap.parse_args()
    for k, v in update(a.workload, a.csv, a.capture, a.json).items():
        print(f"{a.workload} {k}: {sum(v) / len(v) / 1e6:.1f} MB per launch over {len(v)} launches")
