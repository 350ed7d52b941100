"""Writes profiles/traffic.json and a markdown table from raw ncu exports (no hand typing).

    ncu -i <capture>.ncu-rep --page raw --csv > profiles/<name>_raw.csv        (on the machine that has the capture)
    python -m paper_2309_06662_b200.ncu_summary profiles/<name>_raw.csv ... [--json profiles/traffic.json] [--md out.md]

Every row of a raw page is one profiled launch.  Per kernel (demangled name up to the first '(') the launches are averaged.
traffic.json gets, for the workload named by --workload: per-kernel DRAM bytes per launch, warp / thread instructions per
launch, and the sum over one step ("step": kernels x launches per step as given by --per-step name=count ...).
"""
import argparse
import csv
import json
import os
import re
import sys

KEYS = ["gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "launch__grid_size", "launch__block_size",
        "launch__registers_per_thread", "launch__shared_mem_per_block_dynamic", "launch__occupancy_limit_registers",
        "launch__occupancy_limit_shared_mem", "sm__warps_active.avg.pct_of_peak_sustained_active", "smsp__inst_executed.sum",
        "smsp__thread_inst_executed_per_inst_executed.ratio", "smsp__issue_active.avg.pct_of_peak_sustained_active",
        "sm__inst_executed.avg.per_cycle_elapsed", "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
        "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active", "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active",
        "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed", "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum",
        "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "lts__t_sector_hit_rate.pct"]
STALL = re.compile(r"smsp__average_warps?_issue_stalled_(\w+)_per_issue_active\.ratio|smsp__average_warp_latency_issue_stalled_(\w+)\.ratio")
UNIT = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "ms": 1e-3, "us": 1e-6, "ns": 1e-9, "s": 1.0, "msecond": 1e-3,
        "usecond": 1e-6, "nsecond": 1e-9, "second": 1.0}


def short(name):
    return re.sub(r"^void\s+", "", name).split("(")[0].replace("ocn::", "")


def read(path):
    rows = list(csv.reader(open(path)))
    hi = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    hdr, units, data = rows[hi], rows[hi + 1], rows[hi + 2:]
    out = []
    for r in data:
        if len(r) != len(hdr):
            continue
        d = {"kernel": short(r[hdr.index("Kernel Name")])}
        for c, (h, u) in enumerate(zip(hdr, units)):
            try:
                v = float(r[c].replace(",", ""))
            except ValueError:
                continue
            d[h] = v * UNIT[u] if (h.startswith("dram__bytes") or h == "gpu__time_duration.sum") and u in UNIT else v
        out.append(d)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("csv", nargs="+")
    ap.add_argument("--json")
    ap.add_argument("--md")
    ap.add_argument("--workload", default="")
    ap.add_argument("--per-step", nargs="*", default=[], help="kernel-substring=launches per step, for the step total")
    a = ap.parse_args()
    launches = [d for p in a.csv for d in read(p)]
    by = {}
    for d in launches:
        by.setdefault(d["kernel"], []).append(d)
    avg = {k: {h: sum(x.get(h, 0.0) for x in v) / len(v) for h in set().union(*v) if h != "kernel"} for k, v in by.items()}
    lines = ["| kernel | " + " | ".join(k for k in avg) + " |", "|---|" + "---|" * len(avg)]
    stall_names = sorted({h for v in avg.values() for h in v if STALL.match(h)})
    for h in KEYS + stall_names:
        if any(h in v for v in avg.values()):
            lines.append("| `%s` | " % h + " | ".join(("%.6g" % v[h]) if h in v else "" for v in avg.values()) + " |")
    lines.append("| launches averaged | " + " | ".join(str(len(by[k])) for k in avg) + " |")
    text = "\n".join(lines) + "\n"
    if a.md:
        open(a.md, "w").write(text)
    else:
        sys.stdout.write(text)
    if a.json:
        try:
            tj = json.load(open(a.json))
        except Exception:
            tj = {}
        stage = {"k_tendency_tile": "tendency", "k_backsub_correct": "backsub_correct_pressure"}
        step = 0.0
        for k, v in avg.items():
            dram = v.get("dram__bytes_read.sum", 0.0) + v.get("dram__bytes_write.sum", 0.0)
            for sub, name in stage.items():
                if k.startswith(sub):
                    tj[name + ("+ri" if ("+ri" in a.workload) else "")] = {
                        "workload": a.workload, "kernel": k, "dram_bytes_per_launch": dram,
                        "warp_instructions_per_launch": v.get("smsp__inst_executed.sum"),
                        "thread_instructions_per_launch": v.get("smsp__inst_executed.sum", 0.0)
                        * v.get("smsp__thread_inst_executed_per_inst_executed.ratio", 0.0),
                        "source": ", ".join(os.path.basename(p) for p in a.csv)}
            for spec in a.per_step:
                sub, n = spec.split("=")
                if sub in k:
                    step += dram * float(n)
        if a.per_step:
            tj["step" + ("+ri" if ("+ri" in a.workload) else "")] = {
                "workload": a.workload, "dram_bytes_per_step": step, "per_step": a.per_step,
                "source": ", ".join(os.path.basename(p) for p in a.csv)}
        json.dump(tj, open(a.json, "w"), indent=1)


if __name__ == "__main__":
    main()
