"""Records the measured DRAM traffic of the dominant deposit kernel for bench.py's `roofline.traffic`.

    ncu -i gpurun_out/<capture>.ncu-rep --page raw --csv > raw.csv
    python -m paper_1908_02219_b200.profile_traffic raw.csv <workload> [source note]

reads dram__bytes_read.sum + dram__bytes_write.sum of the (first) captured launch and stores them in
profiles/r02_traffic.json under the workload name, together with a hash of the kernel sources: bench.py
reports the figure only while that hash still matches the tree (a capture of older sources is stale).
"""
from __future__ import annotations

import csv
import datetime
import hashlib
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
OUT = os.path.join(ROOT, "profiles", "r02_traffic.json")
KERNEL_SOURCES = ("orb_deposit_ws2.cu", "orb_deposit_ws.cu", "orb_deposit_tile.cu", "orb_geom.cuh")
UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def kernel_source_hash() -> str:
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(HERE, "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def read_raw(path: str):
    rows = list(csv.reader(open(path)))
    hdr, units, vals = rows[0], rows[1], rows[2]
    col = {h: i for i, h in enumerate(hdr)}

    def get(name):
        i = col[name]
        return float(vals[i].replace(",", "")) * UNIT[units[i]]

    kernel = vals[col["Kernel Name"]]
    return kernel, get("dram__bytes_read.sum"), get("dram__bytes_write.sum"), vals[col["gpu__time_duration.sum"]] \
        + " " + units[col["gpu__time_duration.sum"]]


def main(argv):
    raw, workload = argv[1], argv[2]
    note = argv[3] if len(argv) > 3 else os.path.basename(raw)
    kernel, rd, wr, dur = read_raw(raw)
    try:
        db = json.load(open(OUT))
    except Exception:  # noqa: BLE001
        db = {"what": "DRAM bytes of ONE launch of the deposit kernel (ncu --set full); see "
                      "paper_1908_02219_b200/profile_traffic.py", "entries": {}}
    db["entries"][workload] = {
        "kernel": kernel, "dram_bytes_read": int(rd), "dram_bytes_write": int(wr),
        "dram_bytes": int(rd + wr), "duration_under_ncu": dur,
        "kernel_source_sha16": kernel_source_hash(), "source": note,
        "captured": datetime.date.today().isoformat()}
    with open(OUT, "w") as f:
        json.dump(db, f, indent=1, sort_keys=True)
        f.write("\n")
    print(json.dumps(db["entries"][workload]))


if __name__ == "__main__":
    main(sys.argv)
