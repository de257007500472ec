"""Reads `ncu --set full` captures of the sweep kernels and writes the per-launch DRAM traffic bench.py reports.

    python -m paper_1305_3440_b200.profile_traffic OUT.json NAME=REPORT.ncu-rep [NAME=REPORT.ncu-rep ...]
    (REPORT may also be the .csv written by `ncu -i REPORT.ncu-rep --page raw --csv`)

NAME is a bench.py variant (f64-18, f64-12, f32-18, f32-12); NAME@run marks a single-pass capture of consecutive
launches taken with ``--cache-control none`` and only the DRAM byte and duration metrics (no replay, no L2 flush:
the traffic of a launch as it runs inside a step, with the L2 reuse between consecutive half-sweeps), stored under
the variant's "in_run" key.  For every report the launches whose kernel name
contains "sweep" are read with `ncu -i REPORT --page raw --csv` (works without a GPU) and
dram__bytes_read.sum + dram__bytes_write.sum, gpu__time_duration.sum and a few evidence counters are averaged
over them.  The JSON records the hash of the kernel sources (build.source_hash) the library had when this
script ran, i.e. at the code the capture was taken with if it is run right after the capture; bench.py prints
``traffic: null`` when the sources have changed since.  Marshalling of profiler output only.
"""
import csv
import io
import json
import subprocess
import sys

from .build import source_hash

NCU = "/usr/local/cuda/bin/ncu"
WANT = {
    "dram__bytes_read.sum": "dram_read_bytes",
    "dram__bytes_write.sum": "dram_write_bytes",
    "gpu__time_duration.sum": "duration_us",
    "launch__registers_per_thread": "registers",
    "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active": "fp64_pipe_pct",
    "smsp__issue_active.avg.pct_of_peak_sustained_active": "issue_active_pct",
    "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed": "dram_throughput_pct",
    "lts__t_sector_hit_rate.pct": "l2_hit_pct",
    "sm__warps_active.avg.pct_of_peak_sustained_active": "warps_active_pct",
    "smsp__inst_executed.sum": "warp_instructions",
}
SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "us": 1.0, "ms": 1e3, "ns": 1e-3, "s": 1e6,
         "usecond": 1.0, "msecond": 1e3, "nsecond": 1e-3, "second": 1e6}


def read_report(path, pattern="sweep"):
    if path.endswith(".csv"):               # already exported with `ncu -i REPORT --page raw --csv > path`
        out = open(path).read()
    else:
        out = subprocess.run([NCU, "-i", path, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    header, units, data = rows[0], rows[1], rows[2:]
    col = {name: i for i, name in enumerate(header)}
    launches = [r for r in data if pattern in r[col["Kernel Name"]]]
    if not launches:
        raise SystemExit("%s: no launch matches %r" % (path, pattern))
    res = {"kernel": launches[0][col["Kernel Name"]], "launches": len(launches)}
    for metric, key in WANT.items():
        if metric not in col:
            continue
        scale = SCALE.get(units[col[metric]], 1.0)
        vals = [float(r[col[metric]].replace(",", "")) * scale for r in launches]
        res[key] = sum(vals) / len(vals)
    res["traffic_bytes"] = res["dram_read_bytes"] + res["dram_write_bytes"]
    return res


def main(argv):
    if len(argv) < 3 or any("=" not in a for a in argv[2:]):
        raise SystemExit(__doc__)
    doc = {"source_hash": source_hash(), "how": "ncu --set full --clock-control none, averaged over the captured sweep launches "
           "(see the .md beside this file for the command)", "variants": {}}
    for a in sorted(argv[2:], key=lambda a: "@run" in a):
        name, path = a.split("=", 1)
        if name.endswith("@run"):
            doc["variants"].setdefault(name[:-4], {})["in_run"] = read_report(path)
        else:
            doc["variants"][name] = read_report(path)
    json.dump(doc, open(argv[1], "w"), indent=1, sort_keys=True)
    print(json.dumps(doc, indent=1, sort_keys=True))


if __name__ == "__main__":
    main(sys.argv)
