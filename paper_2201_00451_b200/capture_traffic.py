"""Writes `paper_2201_00451_b200/traffic_table.csv`: the DRAM bytes per template of the two FFT kernels, per FFT length,
measured by ncu on a B200 -- the table `bench.py` multiplies by its own CUDA-event times for `roofline.traffic`,
`roofline.dram_frac` and the config-3 `dram_*` fractions.

    python -m paper_2201_00451_b200.capture_traffic            (on the GPU box, i.e. under gpurun; about 5 minutes)

For config 2 and one config-3 cell per FFT length 2^15 .. 2^23 it runs

    ncu --metrics dram__bytes_read.sum,dram__bytes_write.sum,gpu__time_duration.sum --clock-control none -k regex:fft_pass \\
        --csv --log-file <raw.csv> python bench.py --workload <w> --steps 1 --warmup 3 --no-e2e --no-cpu-baseline \\
        --no-cufft-compare --no-config3 --no-extra

(3 warm-up steps + 1 timed + 1 profiled step: five identical steps), sums read and write bytes over the launches of the
LAST step per kernel class and divides by the templates of the step.  Every row carries the commit of the tree it was
captured on (`git rev-parse --short HEAD`, or the value of --commit when the tree on the GPU box has no .git); bench.py
prints it in `roofline.traffic_source`, so a reader can tell whether the table describes the kernels being timed.
The raw ncu logs stay in gpurun_out/ (scratch)."""
from __future__ import annotations

import argparse
import csv
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
TABLE = os.path.join(HERE, "traffic_table.csv")
WORKLOADS = ["config3:1:0.1", "config3:2:0.1", "config3:1:0.5", "config3:1:1.0", "config3:1:2.0", "config3:2:2.0",
             "config3:5:2.0", "config3:10:2.0", "config3:20:2.0", "config2"]       # config 2 last: its 2^21 row is the one bench.py's headline uses
N_STEPS = 5          # warm-up 3 + timed 1 + profiled 1


def parse(raw_path):
    """[(kernel name, grid, {metric: value})] per launch, in launch order."""
    rows, launches = [], {}
    with open(raw_path) as f:
        lines = [ln for ln in f if ln.startswith('"')]
    for r in csv.DictReader(lines):
        i = int(r["ID"])
        if i not in launches:
            launches[i] = (r["Kernel Name"], r["Grid Size"], {})
            rows.append(launches[i])
        launches[i][2][r["Metric Name"]] = (float(r["Metric Value"].replace(",", "")), r["Metric Unit"])
    return rows


def to_bytes(v):
    val, unit = v
    return val * {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(unit, 1.0)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--commit", default="")
    ap.add_argument("--raw-dir", default=os.path.join(ROOT, "gpurun_out"))
    ap.add_argument("--out", default=TABLE, help="where to write the table (under gpurun only gpurun_out/ comes back: write it there and copy it)")
    a = ap.parse_args()
    commit = a.commit
    if not commit:
        try:
            commit = subprocess.check_output(["git", "rev-parse", "--short", "HEAD"], cwd=ROOT, text=True).strip()
        except Exception:
            commit = "unknown"
    os.makedirs(a.raw_dir, exist_ok=True)
    sys.path.insert(0, ROOT)
    import bench
    out = []
    for w in WORKLOADS:
        raw = os.path.join(a.raw_dir, "traffic_raw_" + w.replace(":", "_") + ".csv")
        cmd = ["ncu", "--metrics", "dram__bytes_read.sum,dram__bytes_write.sum,gpu__time_duration.sum", "--clock-control", "none",
               "-k", "regex:fft_pass", "--csv", "--log-file", raw, sys.executable, os.path.join(ROOT, "bench.py"), "--workload", w,
               "--steps", "1", "--warmup", "3", "--no-e2e", "--no-cpu-baseline", "--no-cufft-compare", "--no-config3", "--no-extra"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise SystemExit(f"ncu failed on {w}:\n{r.stdout[-2000:]}\n{r.stderr[-2000:]}")
        p = bench.make_workload(w)
        n_t, n_fft = len(p.templates), p.n_fft
        del p
        launches = parse(raw)
        for cls in ("fft_pass1", "fft_pass2"):
            mine = [x for x in launches if (cls + "_kernel<") in x[0]]
            assert mine and len(mine) % N_STEPS == 0, (w, cls, len(mine))
            last = mine[-(len(mine) // N_STEPS):]
            rd = sum(to_bytes(x[2]["dram__bytes_read.sum"]) for x in last) / n_t
            wr = sum(to_bytes(x[2]["dram__bytes_write.sum"]) for x in last) / n_t
            us = sum(x[2]["gpu__time_duration.sum"][0] for x in last) / 1e3 / n_t
            name = last[0][0].split("(")[0].replace("void ", "")
            out.append((cls, n_fft, int(round(rd)), int(round(wr)), commit,
                        f"{w}: {name} grid {last[0][1]}; {len(last)} launch(es) per step; {us:.2f} us per template under ncu"))
            print(out[-1], flush=True)
    with open(a.out, "w") as f:
        f.write("kernel_class,n_fft,dram_read_bytes_per_template,dram_write_bytes_per_template,commit,source\n")
        for row in out:
            f.write(",".join(str(c).replace(",", ";") for c in row) + "\n")
    print("wrote", a.out)


if __name__ == "__main__":
    main()
