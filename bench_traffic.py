#!/usr/bin/env python
"""bench_traffic.py -- turn an `ncu --set full` report of a bench.py run into profiles/traffic.json.

bench.py cannot measure DRAM traffic inside a timed run; its `roofline.traffic` field comes from this file,
and only while the CUDA sources still hash to the value recorded here (otherwise bench.py prints
`traffic: null, traffic_stale: true`).  Usage, on the GPU box (one ncu run per config / variant):

    python bench.py --config 2 --steps 4 --warmup 3 --no-e2e --no-cpu-baseline &&
    ncu --set full --clock-control none -k regex:"fwd_cl_kernel|bwd_pull_kernel" -s 6 -c 2 -o gpurun_out/prof -f \
        python bench.py --config 2 --steps 4 --warmup 3 --no-e2e --no-cpu-baseline
    python bench_traffic.py gpurun_out/prof.ncu-rep --config 2 --variant cl:auto:reuse

(needs the `ncu` command line tool to read the report; no GPU).
"""
import argparse
import csv
import io
import json
import os
import subprocess

ROOT = os.path.dirname(os.path.abspath(__file__))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--variant", default="cl:auto:reuse", help="layout:backward:reuse|noreuse, as bench.py names it")
    args = ap.parse_args()
    from bench import source_hash
    raw = subprocess.run(["ncu", "-i", args.report, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(raw)))
    hdr, units = rows[0], rows[1]
    name, rd, wr, dur = (hdr.index(k) for k in ("Kernel Name", "dram__bytes_read.sum", "dram__bytes_write.sum",
                                                "gpu__time_duration.sum"))
    scale = {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    entry = {}
    for r in rows[2:]:
        leg = "fwd" if "fwd_" in r[name] else ("bwd" if "bwd_" in r[name] else None)
        if leg is None:
            continue
        entry[leg] = int(float(r[rd]) * scale[units[rd]] + float(r[wr]) * scale[units[wr]])
        entry[leg + "_kernel"] = r[name].split("(")[0]
        entry[leg + "_gpu_time_us"] = float(r[dur])
    path = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        t = json.load(open(path))
    except Exception:
        t = {}
    h = source_hash()
    if t.get("source_hash") != h:
        t = {"source_hash": h, "configs": {}}
    t["what"] = "dram__bytes_read.sum + dram__bytes_write.sum per launch, from ncu --set full (see bench_traffic.py)"
    t["configs"][f"{args.config}:{args.variant}"] = entry
    json.dump(t, open(path, "w"), indent=1, sort_keys=True)
    print(json.dumps(entry))


if __name__ == "__main__":
    main()
