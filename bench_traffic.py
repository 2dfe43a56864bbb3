#!/usr/bin/env python
"""bench_traffic.py -- turns one `ncu --set full` capture into the tracked summary bench.py reads.

    python bench_traffic.py <capture.ncu-rep> --workload <config.workload> --name <profiles/ stem> --command "<ncu command line>"

Reads the capture with `ncu -i <rep> --page raw --csv` (works without a GPU), writes `profiles/<name>.md` (the command, one
column per captured launch, the metrics DESIGN.md quotes, every stall reason above 0.05 per issue) and records, per kernel,
`dram__bytes_read.sum + dram__bytes_write.sum` of its LAST captured launch in `profiles/traffic.json` together with the hash
of the kernel sources at the time (bench.kernel_sources_sha): bench.py reports `roofline.traffic` from that file and refuses
an entry whose hash differs from the sources it runs.  Nothing here touches the GPU or the oracle.
"""
from __future__ import annotations

import argparse
import csv
import datetime
import io
import json
import os
import subprocess

import bench

ROOT = os.path.dirname(os.path.abspath(__file__))
WANT = ["gpu__time_duration.sum", "launch__grid_size", "launch__block_size", "launch__registers_per_thread",
        "launch__shared_mem_per_block_dynamic", "launch__occupancy_limit_registers", "launch__occupancy_limit_shared_mem",
        "sm__warps_active.avg.pct_of_peak_sustained_active", "dram__bytes_read.sum", "dram__bytes_write.sum",
        "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "lts__t_sector_hit_rate.pct",
        "l1tex__m_xbar2l1tex_read_bytes.sum", "sm__throughput.avg.pct_of_peak_sustained_elapsed",
        "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
        "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
        "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active",
        "smsp__inst_executed.sum", "smsp__warps_active.avg.per_cycle_active", "smsp__warps_eligible.avg.per_cycle_active",
        "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
        "sm__cycles_active.avg", "sm__cycles_elapsed.max"]
UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def short(name):
    name = name.split("(")[0].replace("void ", "")
    return name.replace("e3::", "").split("<")[0]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("rep")
    ap.add_argument("--workload", required=True)
    ap.add_argument("--name", required=True)
    ap.add_argument("--command", required=True)
    ap.add_argument("--note", default="")
    a = ap.parse_args()
    raw = subprocess.run(["ncu", "-i", a.rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(raw)))
    hdr, units, data = rows[0], rows[1], rows[2:]
    names = [short(r[hdr.index("Kernel Name")]) for r in data]
    sha = bench.kernel_sources_sha()
    lines = [f"# {a.name}: `ncu --set full` of config `{a.workload}`", "",
             "Command (on the B200 box, through `gpurun`; the same command exited 0 without ncu first):", "",
             f"    {a.command}", "", f"Kernel sources hash (bench.kernel_sources_sha): `{sha}`.  {a.note}", "",
             "| metric | unit | " + " | ".join(f"`{n}`" for n in names) + " |", "|---|---|" + "---|" * len(names)]
    for m in WANT:
        if m in hdr:
            i = hdr.index(m)
            lines.append(f"| `{m}` | {units[i]} | " + " | ".join(r[i] for r in data) + " |")
    for i, m in enumerate(hdr):
        if "issue_stalled" in m and m.endswith("per_issue_active.ratio") and "not_issued" not in m:
            vals = [float(r[i] or 0) for r in data]
            vals = [0.0 if v != v else v for v in vals]
            if max(vals) > 0.05:
                lines.append(f"| `{m}` | inst | " + " | ".join(f"{v:.2f}" for v in vals) + " |")
    out_md = os.path.join(ROOT, "profiles", a.name + ".md")
    open(out_md, "w").write("\n".join(lines) + "\n")
    tj = os.path.join(ROOT, "profiles", "traffic.json")
    traffic = json.load(open(tj)) if os.path.exists(tj) else {}
    ir, iw = hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
    it = hdr.index("gpu__time_duration.sum")
    ent = traffic.setdefault(a.workload, {})
    for r, n in zip(data, names):
        b = float(r[ir]) * UNIT_SCALE[units[ir]] + float(r[iw]) * UNIT_SCALE[units[iw]]
        if b != b:             # ncu could not collect this launch's memory counters (NaN in the report): no entry, bench.py reports null
            ent.pop(n, None)
            continue
        ent[n] = {"dram_bytes": int(b), "dram_read_bytes": int(float(r[ir]) * UNIT_SCALE[units[ir]]),
                  "dram_write_bytes": int(float(r[iw]) * UNIT_SCALE[units[iw]]), "duration": f"{r[it]} {units[it]}",
                  "capture": f"profiles/{a.name}.md", "csrc_sha": sha,
                  "captured": datetime.datetime.now(datetime.timezone.utc).strftime("%Y-%m-%d")}
    json.dump(traffic, open(tj, "w"), indent=1, sort_keys=True)
    print(out_md, tj)


if __name__ == "__main__":
    main()
