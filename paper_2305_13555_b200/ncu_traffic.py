"""Measured DRAM traffic of the dominant kernel -> profiles/traffic.json (read by bench.py's `roofline.traffic`).

    python -m paper_2305_13555_b200.ncu_traffic --rep gpurun_out/r2_prof_cfg3.ncu-rep --kernel 'oci_red_resident_kernel<64, 1>' \\
        --entry cfg3_reduced --iterations 6 --capture profiles/r2_reduced_cfg3_full.txt

Reads an `ncu --set full` report with `ncu -i <rep> --page raw --csv`, averages dram__bytes_read.sum +
dram__bytes_write.sum over the launches whose name contains --kernel, divides by --iterations (the fused ITER launches
run all iterations of a time step) and records the result together with the git commit the working tree is at, so a
capture that is older than the kernel it describes is visible next to the number.  No GPU needed."""
import argparse
import csv
import io
import json
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TO_BYTES = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}


def dram_bytes_per_launch(rep, kernel):
    out = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    hdr, units = rows[0], rows[1]
    name = hdr.index("Kernel Name")
    rd, wr, tm = hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum"), hdr.index("gpu__time_duration.sum")
    vals, times = [], []
    for r in rows[2:]:
        if kernel in r[name]:
            vals.append(float(r[rd].replace(",", "")) * TO_BYTES[units[rd]] + float(r[wr].replace(",", "")) * TO_BYTES[units[wr]])
            times.append(float(r[tm].replace(",", "")))
    if not vals:
        raise SystemExit(f"no launch of a kernel matching {kernel!r} in {rep}")
    return sum(vals) / len(vals), len(vals), sum(times) / len(times), units[tm]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--rep", required=True)
    ap.add_argument("--kernel", required=True, help="substring of the kernel name as ncu prints it")
    ap.add_argument("--entry", required=True, help="key in traffic.json, e.g. cfg3_reduced")
    ap.add_argument("--iterations", type=float, default=1.0, help="OCI iterations one captured launch runs")
    ap.add_argument("--capture", default=None, help="the committed text summary of the same report")
    a = ap.parse_args()
    b, n, t, tu = dram_bytes_per_launch(a.rep, a.kernel)
    commit = subprocess.run(["git", "rev-parse", "--short", "HEAD"], cwd=ROOT, capture_output=True, text=True).stdout.strip()
    dirty = subprocess.run(["git", "status", "--porcelain", "--", "paper_2305_13555_b200/csrc"], cwd=ROOT, capture_output=True, text=True).stdout.strip()
    path = os.path.join(ROOT, "profiles", "traffic.json")
    data = json.load(open(path)) if os.path.exists(path) else {"entries": {}}
    data["entries"][a.entry] = {"dram_bytes_per_iteration": b / a.iterations, "dram_bytes_per_launch": b, "iterations_per_launch": a.iterations,
                                "launches_averaged": n, "launch_duration": [t, tu], "kernel": a.kernel, "capture": a.capture,
                                "commit": commit + ("-dirty" if dirty else "")}
    with open(path, "w") as f:
        json.dump(data, f, indent=1, sort_keys=True)
        f.write("\n")
    print(json.dumps(data["entries"][a.entry]))


if __name__ == "__main__":
    main()
