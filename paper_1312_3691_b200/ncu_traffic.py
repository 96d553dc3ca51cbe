"""Write profiles/trace_traffic.json from ncu captures (read by bench.py for `roofline.traffic`).

    python -m paper_1312_3691_b200.ncu_traffic C5=gpurun_out/r3_full_C5_raw.csv C2=... --note "..."

Each CSV is the `ncu -i <report> --page raw --csv` export of one `ncu --set full` capture of a bench.py run of that
config.  For the kernel named by --kernel (default k_trace_wf) the script takes the FIRST captured launch and stores
dram__bytes_read.sum + dram__bytes_write.sum in bytes, its duration and the file it came from.  Nothing here runs on the
GPU or touches the library; it only replaces copying numbers by hand.
"""
from __future__ import annotations

import argparse
import csv
import json
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
OUT = os.path.join(ROOT, "profiles", "trace_traffic.json")
UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
        "ns": 1e-6, "us": 1e-3, "ms": 1.0, "s": 1e3, "nsecond": 1e-6, "usecond": 1e-3, "msecond": 1.0, "second": 1e3}


def read_raw_csv(path: str):
    """Rows of an `ncu --page raw --csv` export as dicts; the row after the header holds the units."""
    with open(path, newline="") as f:
        lines = [ln for ln in f if ln.startswith('"')]          # skip ncu's ==PROF== chatter, if any
    rows = list(csv.reader(lines))
    header, units, body = rows[0], rows[1], rows[2:]
    return header, dict(zip(header, units)), [dict(zip(header, r)) for r in body]


def value(row, units, name: str) -> float:
    return float(row[name].replace(",", "")) * UNIT[units[name]]


def launch_traffic(path: str, kernel: str):
    header, units, body = read_raw_csv(path)
    for row in body:
        if kernel in row["Kernel Name"]:
            rd, wr = value(row, units, "dram__bytes_read.sum"), value(row, units, "dram__bytes_write.sum")
            return {"dram_bytes_per_launch": int(round(rd + wr)), "dram_bytes_read": int(round(rd)),
                    "dram_bytes_write": int(round(wr)), "launch_ms_under_ncu": value(row, units, "gpu__time_duration.sum")}
    raise SystemExit(f"{path}: no launch of {kernel}")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("captures", nargs="+", help="CONFIG=raw.csv")
    ap.add_argument("--kernel", default="k_trace_wf")
    ap.add_argument("--note", default="", help="what the captures were (command, which launch), stored as `source`")
    args = ap.parse_args()
    out = json.load(open(OUT)) if os.path.exists(OUT) else {}
    for item in args.captures:
        cfg, path = item.split("=", 1)
        d = launch_traffic(path, args.kernel)
        d["source"] = f"{os.path.basename(path)}: {args.note}".strip(": ")
        out[cfg] = d
    with open(OUT, "w") as f:
        json.dump(out, f, indent=1, sort_keys=True)
        f.write("\n")
    print(json.dumps(out, indent=1, sort_keys=True))


if __name__ == "__main__":
    main()
