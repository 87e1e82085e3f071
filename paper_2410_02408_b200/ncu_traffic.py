"""Writes profiles/traffic.txt from committed ncu raw exports (no hand transcription).

An export is the text of `ncu -i <capture>.ncu-rep --page raw --csv --print-units base` of an
`ncu --set full --clock-control none` capture of `bench.py --config C [--block B] --no-extras`
(the full commands are named in the .md beside each .csv under profiles/).  For every kernel of the
operator path the script takes dram__bytes_read.sum + dram__bytes_write.sum per launch (mean over the
captured launches of that kernel kind) -- the `traffic` figure of bench.py's roofline object.

    python -m paper_2410_02408_b200.ncu_traffic cfg2_b8=profiles/r2_ncu_raw_cfg2_b8.csv [cfg3_b32=...] > profiles/traffic.txt
"""
from __future__ import annotations

import csv
import json
import re
import sys


def kernel_kind(name: str):
    """bench.py's kernel-kind key for a (demangled) kernel name, or None for kernels outside the operator apply."""
    m = re.search(r"(\w+)<([^>]*)>", name)
    base = m.group(1) if m else name.split("(")[0].split()[-1]
    targs = [a.strip() for a in m.group(2).split(",")] if m else []

    def arg(i):
        a = targs[i].split(")")[-1]          # "(bool)1" style casts
        return {"true": 1, "false": 0}.get(a, None) if a in ("true", "false") else int(a)

    dirs = {0: "solve_L", 1: "solve_Lt", 2: "apply"}
    if base == "spmv_stream_kernel":
        return "spmv_solve_L" if arg(1) == 1 else "spmv"
    if base in ("spmv_vector_kernel", "spmv_bsr3_kernel"):
        return "spmv"
    if base == "solve_small_kernel":
        return dirs[arg(1)]
    if base in ("solve_group_kernel", "solve_band_kernel"):
        return dirs[arg(2)]
    if base == "solve_stream_kernel":
        return dirs[arg(1)]
    if base == "solve_var_kernel":
        return dirs[arg(0)]
    return None


def read_export(path: str) -> dict:
    """{kind: {"launches", "dram_bytes", "dram_read", "dram_write", "us", "kernel"}} from one raw CSV export."""
    with open(path, newline="") as fh:
        rows = [r for r in csv.reader(fh) if r]
    hdr = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    cols = {c: k for k, c in enumerate(rows[hdr])}
    units = rows[hdr + 1]
    need = ("dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__time_duration.sum")
    for c in need:
        if c not in cols:
            raise SystemExit(f"{path}: column {c} missing (export with --page raw --csv of a --set full capture)")
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "ns": 1e-3, "us": 1.0, "usecond": 1.0, "nsecond": 1e-3,
             "msecond": 1e3, "ms": 1e3}

    def val(r, c):
        return float(r[cols[c]].replace(",", "")) * scale.get(units[cols[c]], 1.0)

    acc = {}
    for r in rows[hdr + 2:]:
        kind = kernel_kind(r[cols["Kernel Name"]])
        if kind is None:
            continue
        a = acc.setdefault(kind, {"launches": 0, "dram_read": 0.0, "dram_write": 0.0, "us": 0.0, "kernel": r[cols["Kernel Name"]].split("(")[0]})
        a["launches"] += 1
        a["dram_read"] += val(r, "dram__bytes_read.sum")
        a["dram_write"] += val(r, "dram__bytes_write.sum")
        a["us"] += val(r, "gpu__time_duration.sum")
    for a in acc.values():
        k = a["launches"]
        a["dram_read"], a["dram_write"], a["us"] = a["dram_read"] / k, a["dram_write"] / k, a["us"] / k
        a["dram_bytes"] = a["dram_read"] + a["dram_write"]
    return acc


def main(argv):
    out = {"_comment": "dram__bytes_read.sum + dram__bytes_write.sum per launch (bytes), written by "
                       "`python -m paper_2410_02408_b200.ncu_traffic` from the ncu raw exports named in _sources", "_sources": {}}
    for item in argv:
        key, path = item.split("=", 1)
        out["_sources"][key] = path
        out[key] = {kind: int(round(a["dram_bytes"])) for kind, a in sorted(read_export(path).items())}
    json.dump(out, sys.stdout, indent=1)
    sys.stdout.write("\n")


if __name__ == "__main__":
    main(sys.argv[1:])
