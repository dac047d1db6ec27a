"""Measurement bookkeeping for bench.py's `roofline.traffic` (no method arithmetic).

`kernel_sources_hash()` identifies the kernel sources a DRAM-traffic figure was
captured from (the gather sweeps of the headline path and the table layout they
walk); bench.py attaches a stored figure only while the hash still matches.  Run as a module to turn one `ncu --set full` capture into
profiles/ncu_traffic.json:

    ncu -i gpurun_out/prof.ncu-rep --page raw --csv > raw.csv
    python -m paper_1204_3425_b200.ncu_traffic raw.csv --config C4 --dtype f64 \
        --command "<the ncu command that made the capture>" [--append]

Kernel names are mapped to bench.py's kernel classes: gather_sweep_kernel<..., COL = 0/1, ...> -> row_sweep /
col_sweep, strip_sweep_kernel -> col_sweep, row_* -> row_sweep, hv_paper_kernel -> hv_paper.
"""
from __future__ import annotations

import csv
import hashlib
import json
import sys
import time
from pathlib import Path

PKG = Path(__file__).resolve().parent
OUT = PKG.parent / "profiles" / "ncu_traffic.json"


# what decides the DRAM traffic of the captured kernels: the gather sweeps, their reductions, the table layout
HASHED = ("kernels_gather.cuh", "kernels_common.cuh", "gather_tables.cpp", "gather_tables.h")


def kernel_sources_hash() -> str:
    h = hashlib.sha256()
    for name in HASHED:
        h.update(name.encode())
        h.update((PKG / "csrc" / name).read_bytes())
    return h.hexdigest()


def kclass_of(kernel: str) -> str | None:
    if "gather_sweep_kernel" in kernel:
        # template arguments <T, R, E, COL, LZ>: ncu prints bools as 0/1 (or false/true)
        args = kernel[kernel.index("<") + 1:kernel.rindex(">")].split(",")
        col = args[3].strip().lstrip("(bool)") in ("1", "true")
        return "col_sweep" if col else "row_sweep"
    if "strip_sweep_kernel" in kernel:
        return "col_sweep"
    if "row_" in kernel and "kernel" in kernel:
        return "row_sweep"
    if "hv_paper_kernel" in kernel:
        return "hv_paper"
    if "axpy_norm" in kernel:
        return "vec_sweep"
    return None


def parse_raw_csv(path: str):
    """Per kernel name: mean of dram__bytes_read.sum + dram__bytes_write.sum over the captured launches."""
    rows = list(csv.reader(open(path, newline="")))
    hdr = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    names, units = rows[hdr], rows[hdr + 1]
    k_name = names.index("Kernel Name")
    k_rd, k_wr = names.index("dram__bytes_read.sum"), names.index("dram__bytes_write.sum")
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    acc = {}
    for r in rows[hdr + 2:]:
        if len(r) <= max(k_rd, k_wr):
            continue
        b = float(r[k_rd].replace(",", "")) * scale[units[k_rd]] + float(r[k_wr].replace(",", "")) * scale[units[k_wr]]
        acc.setdefault(r[k_name], []).append(b)
    return {k: sum(v) / len(v) for k, v in acc.items()}


def main(argv):
    import argparse
    p = argparse.ArgumentParser()
    p.add_argument("raw_csv")
    p.add_argument("--config", required=True)
    p.add_argument("--dtype", required=True)
    p.add_argument("--command", required=True)
    p.add_argument("--append", action="store_true", help="keep the entries of other (config, dtype) pairs")
    a = p.parse_args(argv)
    h = kernel_sources_hash()
    rec = {"entries": []}
    if a.append and OUT.exists():
        old = json.loads(OUT.read_text())
        if old.get("kernel_sources_sha256") == h:
            rec = old
    rec["kernel_sources_sha256"] = h
    rec["captured"] = time.strftime("%Y-%m-%d")
    rec.setdefault("commands", {})[f"{a.config}/{a.dtype}"] = a.command
    rec["entries"] = [e for e in rec["entries"] if (e["config"], e["dtype"]) != (a.config, a.dtype)]
    for kernel, b in parse_raw_csv(a.raw_csv).items():
        kc = kclass_of(kernel)
        if kc:
            rec["entries"].append({"config": a.config, "dtype": a.dtype, "kclass": kc, "kernel": kernel,
                                   "dram_bytes_per_launch": b})
    OUT.write_text(json.dumps(rec, indent=1) + "\n")
    print(f"wrote {OUT} ({len(rec['entries'])} entries, sources {h[:12]})")


if __name__ == "__main__":
    main(sys.argv[1:])
