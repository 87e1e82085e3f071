"""Writes profiles/traffic.txt from committed ncu raw exports (no hand transcription).

An export is the text of `ncu -i <capture>.ncu-rep --page raw --csv --print-units base` of an
`ncu --set full --clock-control none` capture of `bench.py --config C [--block B] --no-extras`
(the full commands are named in the .md beside each .csv under profiles/).  For every kernel of the
operator path the script takes dram__bytes_read.sum + dram__bytes_write.sum per launch (mean over the
captured launches of that kernel kind) -- the `traffic` figure of bench.py's roofline object.

    python -m paper_2410_02408_b200.ncu_traffic cfg2_b8=profiles/r2_ncu_raw_cfg2_b8.csv [cfg3_b32=...] > profiles/traffic.txt
    python -m paper_2410_02408_b200.ncu_traffic --summary cfg2_b8=... [...] > profiles/r2_ncu_full.md     (the table of counters)
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


SUMMARY_METRICS = [
    ("gpu__time_duration.sum", "duration (us)", 1e-3), ("dram__bytes_read.sum", "DRAM read (MB)", 1e-6),
    ("dram__bytes_write.sum", "DRAM write (MB)", 1e-6),
    ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "DRAM throughput (% of ncu peak)", 1),
    ("l1tex__m_xbar2l1tex_read_bytes.sum", "L2 -> L1 bytes (MB)", 1e-6), ("l1tex__t_sector_hit_rate.pct", "L1 sector hit (%)", 1),
    ("lts__t_sector_hit_rate.pct", "L2 sector hit (%)", 1), ("sm__warps_active.avg.pct_of_peak_sustained_active", "warps active (% of peak)", 1),
    ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue active (%)", 1), ("launch__registers_per_thread", "registers / thread", 1),
    ("launch__grid_size", "grid", 1), ("launch__block_size", "block", 1), ("launch__shared_mem_per_block_dynamic", "dynamic smem / CTA (KB)", 1e-3)]
SHAPES = {"cfg2": (2097152, 14581760), "cfg3": (1048576, 17825676), "cfg4": (4194304, 37724164), "cfg5": (2654208, 210542904)}


def algorithmic(key: str, kind: str) -> int:
    """Byte count of DESIGN.md section 5 / SURVEY.md 8(d) for a kernel kind of `cfgC_bB`."""
    cfg, b = key.split("_b")
    n, nnz = SHAPES[cfg]
    b = int(b)
    spmv, solve = 12 * nnz + 4 * (n + 1) + 16 * n, 4 * n * (b + 1) + 16 * n
    return {"spmv": spmv, "solve_L": solve, "solve_Lt": solve, "apply": solve, "spmv_solve_L": spmv + solve}[kind]


def summary(argv):
    """Markdown table of the counters per kernel kind (means over the captured launches) for each `key=path`."""
    w = sys.stdout.write
    w("# ncu `--set full`, the kernels of `bj_op_apply` (rotating inputs)\n\n")
    w("Commands (per config C, block B; after the plain run of the same command exited 0 in the same call):\n\n```\n")
    w("ncu --set full --clock-control none --import-source on -k regex:\"spmv_stream|solve_small|solve_group\" -s 40 -c 6 \\\n")
    w("    -o prof python bench.py --config C --block B --steps 20 --warmup 5 --no-extras\n")
    w("ncu -i prof.ncu-rep --page raw --csv --print-units base > profiles/r2_ncu_raw_cfgC_bB.csv\n")
    w("python -m paper_2410_02408_b200.ncu_traffic --summary " + " ".join(argv) + "\n```\n\n")
    w("Means over the captured launches of each kernel kind; the raw exports are beside this file.  `algorithmic` = the byte count of\n"
      "DESIGN.md section 5 / SURVEY.md 8(d); `DRAM / algorithmic` < 1: vectors (and, in a chain of applies, the serpentine factor slice)\n"
      "came from L2; `L2 -> L1 / algorithmic` > 1: sector over-fetch (config 3's 8-byte gathers pull 32-byte sectors).\n\n")
    for item in argv:
        key, path = item.split("=", 1)
        with open(path, newline="") as fh:
            rows = [r for r in csv.reader(fh) if r]
        hdr = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
        col = {c: k for k, c in enumerate(rows[hdr])}
        acc = {}
        for r in rows[hdr + 2:]:
            kind = kernel_kind(r[col["Kernel Name"]])
            if kind is None:
                continue
            a = acc.setdefault(kind, {"name": r[col["Kernel Name"]].split("(")[0].replace("void ", "").replace("unnamed>::", ""), "n": 0})
            a["n"] += 1
            for m, _, _ in SUMMARY_METRICS:
                a[m] = a.get(m, 0.0) + float(r[col[m]].replace(",", ""))
        kinds = [k for k in ("solve_Lt", "spmv", "spmv_solve_L", "solve_L", "apply") if k in acc]
        mean = lambda k, m: acc[k][m] / acc[k]["n"]  # noqa: E731
        n, nnz = SHAPES[key.split("_b")[0]]
        w(f"## {key}  (N = {n}, nnz = {nnz}, b = {key.split('_b')[1]})\n\n")
        w("| metric | " + " | ".join(f"{k}: `{acc[k]['name']}`" for k in kinds) + " |\n|---|" + "---|" * len(kinds) + "\n")
        for m, label, sc in SUMMARY_METRICS:
            w(f"| {label} | " + " | ".join("%.1f" % (mean(k, m) * sc) for k in kinds) + " |\n")
        w("| algorithmic bytes (MB) | " + " | ".join("%.1f" % (algorithmic(key, k) / 1e6) for k in kinds) + " |\n")
        w("| DRAM / algorithmic | " + " | ".join(
            "%.2f" % ((mean(k, "dram__bytes_read.sum") + mean(k, "dram__bytes_write.sum")) / algorithmic(key, k)) for k in kinds) + " |\n")
        w("| L2 -> L1 / algorithmic | " + " | ".join(
            "%.2f" % (mean(k, "l1tex__m_xbar2l1tex_read_bytes.sum") / algorithmic(key, k)) for k in kinds) + " |\n")
        w("| algorithmic GB/s under ncu (cold, serialised) | " + " | ".join(
            "%.0f" % (algorithmic(key, k) / mean(k, "gpu__time_duration.sum")) for k in kinds) + " |\n\n")


def main(argv):
    if argv and argv[0] == "--summary":
        return summary(argv[1:])
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
