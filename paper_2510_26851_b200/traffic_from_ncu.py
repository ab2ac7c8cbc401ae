"""python -m paper_2510_26851_b200.traffic_from_ncu REPORT.ncu-rep --workload cfg2 > profiles/traffic.json

Turns one `ncu --set full` capture into the `traffic` figures bench.py prints: per stage of the path, the mean of
dram__bytes_read.sum + dram__bytes_write.sum per launch of its kernel.  The output also carries a hash of the CUDA
sources the capture was taken from; bench.py recomputes it and prints `traffic: null` when the sources have
changed since (a number from another tree is not a measurement of this one)."""
from __future__ import annotations

import argparse
import csv
import hashlib
import json
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")

# kernel name (substring) -> profiled stage of fof_profile_name()
KERNEL_STAGE = {
    "part_hist_kernel": "link.hist", "part_offsets_kernel": "link.offsets", "part_scatter_kernel": "link.partition",
    "cell_sort_kernel": "link.cell_sort", "link_kernel": "link.pairs", "write_labels_kernel": "link.labels",
    "group_count_kernel": "groups.count", "group_compact_kernel": "groups.compact",
    "group_reduce_kernel": "groups.reduce", "group_finish_kernel": "groups.finish",
    "block_scatter_kernel": "block.partition", "block_link_kernel": "block.link",
    "cross_link_kernel": "block.cross", "flatten_labels_kernel": "block.flatten",
}
UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def source_hash() -> str:
    """sha256 over the CUDA sources of the library, in name order (first 16 hex digits)."""
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh")):
            with open(os.path.join(CSRC, name), "rb") as f:
                h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--command", default="", help="the command line the capture was made with (recorded verbatim)")
    a = ap.parse_args()
    out = subprocess.run(["ncu", "-i", a.report, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(out.splitlines()))
    hdr, units = rows[0], rows[1]
    ik, ir, iw, it = (hdr.index(c) for c in ("Kernel Name", "dram__bytes_read.sum", "dram__bytes_write.sum",
                                               "gpu__time_duration.sum"))
    acc: dict[str, list] = {}
    for r in rows[2:]:
        stage = next((s for k, s in KERNEL_STAGE.items() if k + "<" in r[ik] or k + "(" in r[ik]), None)
        if stage is None:
            continue
        b = float(r[ir].replace(",", "")) * UNIT[units[ir]] + float(r[iw].replace(",", "")) * UNIT[units[iw]]
        e = acc.setdefault(stage, [0, 0.0, 0.0])
        e[0] += 1; e[1] += b; e[2] += float(r[it].replace(",", ""))
    doc = {"source_hash": source_hash(), "report": os.path.basename(a.report), "command": a.command,
           "what": "dram__bytes_read.sum + dram__bytes_write.sum per launch (mean over the captured launches), bytes",
           a.workload: {s: int(round(e[1] / e[0])) for s, e in sorted(acc.items())},
           a.workload + "_launches": {s: e[0] for s, e in sorted(acc.items())},
           a.workload + "_ncu_us": {s: round(e[2] / e[0], 2) for s, e in sorted(acc.items())}}
    json.dump(doc, sys.stdout, indent=1)
    print()


if __name__ == "__main__":
    main()
