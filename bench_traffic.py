#!/usr/bin/env python
"""bench_traffic.py -- turn one `ncu --set full` capture of the two FFT-pass kernels into the tracked
summary profiles/traffic.json that bench.py reads for `roofline.traffic`.

On the GPU box, in the same gpurun command as the capture (stamps the kernel sources the capture ran on):

    python bench_traffic.py --stamp > gpurun_out/src_hash.txt

Here (CPU box, ncu can read reports without a GPU):

    python bench_traffic.py --report gpurun_out/prof.ncu-rep --stamp-file gpurun_out/src_hash.txt \
        --n 1048576 --templates-per-launch 64 --command "<the ncu command line>"

dram bytes per template = (dram__bytes_read.sum + dram__bytes_write.sum) of a launch / templates per
launch, averaged over the captured launches of each kernel.  bench.py reports `traffic: null` when the
hash stored here is not that of the kernel sources it runs on.
"""
from __future__ import annotations

import argparse
import csv
import io
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--stamp", action="store_true", help="print the hash of the kernel sources and exit")
    ap.add_argument("--report")
    ap.add_argument("--stamp-file")
    ap.add_argument("--n", type=int, default=1 << 20)
    ap.add_argument("--templates-per-launch", type=int, default=64)
    ap.add_argument("--command", default="")
    ap.add_argument("--out", default=os.path.join(ROOT, "profiles", "traffic.json"))
    a = ap.parse_args()
    from bench import kernel_source_hash
    if a.stamp:
        print(kernel_source_hash())
        return 0
    stamp = open(a.stamp_file).read().strip() if a.stamp_file else kernel_source_hash()
    raw = subprocess.run(["ncu", "-i", a.report, "--page", "raw", "--csv"], check=True, capture_output=True, text=True).stdout
    rows = list(csv.reader(io.StringIO(raw)))
    hdr = rows[0]
    col = {name: i for i, name in enumerate(hdr)}
    per = {"p1_kernel": [], "p2_kernel": []}
    dur = {"p1_kernel": [], "p2_kernel": []}
    for r in rows[2:]:                       # row 1 holds the units
        name = r[col["Kernel Name"]]
        for k in per:
            if k in name:
                rd = float(r[col["dram__bytes_read.sum"]].replace(",", ""))
                wr = float(r[col["dram__bytes_write.sum"]].replace(",", ""))
                unit_r = rows[1][col["dram__bytes_read.sum"]]
                unit_w = rows[1][col["dram__bytes_write.sum"]]
                scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
                per[k].append(rd * scale.get(unit_r, 1.0) + wr * scale.get(unit_w, 1.0))
                d = float(r[col["gpu__time_duration.sum"]].replace(",", ""))
                dur[k].append(d * {"ns": 1e-3, "us": 1.0, "ms": 1e3}.get(rows[1][col["gpu__time_duration.sum"]], 1.0))
    out = {
        "kernel_source_hash": stamp, "n": a.n, "templates_per_launch": a.templates_per_launch,
        "launches_captured": [len(per["p1_kernel"]), len(per["p2_kernel"])],
        "dram_bytes_per_template": [sum(v) / len(v) / a.templates_per_launch if v else None for v in (per["p1_kernel"], per["p2_kernel"])],
        "gpu_time_us_per_launch_under_ncu": [sum(v) / len(v) if v else None for v in (dur["p1_kernel"], dur["p2_kernel"])],
        "source": f"ncu --set full, {os.path.basename(a.report)} (profiles/traffic.json)", "command": a.command,
    }
    with open(a.out, "w") as fh:
        json.dump(out, fh, indent=1)
        fh.write("\n")
    print(json.dumps(out))
    return 0


if __name__ == "__main__":
    sys.exit(main())
