#!/usr/bin/env python
"""ncu_summary.py -- turns an Nsight Compute report of bench.py into the text summaries kept under profiles/.

    # on the B200 box (gpurun), after the same bench.py command has exited 0 without ncu:
    ncu --set full --clock-control none --import-source on -k regex:"_kernel" -s <skip> -c <n> \
        -o gpurun_out/<name> -f python bench.py --steps 4 --warmup 3 --no-extras
    # here (no GPU needed):
    python ncu_summary.py gpurun_out/<name>.ncu-rep [--md profiles/<name>.md] [--traffic profiles/<name>_traffic.json]
    python ncu_summary.py --launches gpurun_out/<launch list>.csv          # the gpu__time_duration.sum launch list

The table has one row per captured launch: duration, grid, registers, tensor-pipe busy share, issue-active share, warp
instructions, DRAM bytes read / written (per launch: this is `roofline.traffic` of bench.py), achieved DRAM GB/s, L2 hit
rate.  --traffic writes {"<kernel name>": mean dram bytes per launch} for bench.py to report.
"""
import argparse
import csv
import json
import subprocess
import sys

K_HMMA = "sm__pipe_tensor_subpipe_hmma_cycles_active_realtime.avg"
COLS = ["gpu__time_duration.sum", "launch__grid_size", "launch__registers_per_thread", "smsp__cycles_elapsed.avg",
        "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__warps_active.avg.pct_of_peak_sustained_active",
        "smsp__inst_executed.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "lts__t_sector_hit_rate.pct"]


def short(name):
    n = name.replace("<unnamed>::", "").replace("void ", "")
    for cut in ("(<", "(const", "(int", "("):
        if cut in n:
            n = n.split(cut)[0]
    return n


def raw_rows(rep):
    out = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(out.splitlines()))
    hdr, units = rows[0], rows[1]
    return hdr, units, rows[2:]


def to_float(v):
    try:
        return float(v.replace(",", ""))
    except ValueError:
        return float("nan")


def summarise(rep):
    hdr, units, rows = raw_rows(rep)
    ci = {h: i for i, h in enumerate(hdr)}
    hm = [h for h in hdr if h.endswith(K_HMMA)]
    table = []
    for r in rows:
        g = lambda k: to_float(r[ci[k]]) if k in ci else float("nan")
        unit = lambda k: units[ci[k]] if k in ci else ""
        t = g("gpu__time_duration.sum")
        t_us = t / 1e3 if unit("gpu__time_duration.sum") in ("ns", "nsecond") else (t if unit("gpu__time_duration.sum") in ("us", "usecond") else t)
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
        dr = g("dram__bytes_read.sum") * scale.get(unit("dram__bytes_read.sum"), 1.0)
        dw = g("dram__bytes_write.sum") * scale.get(unit("dram__bytes_write.sum"), 1.0)
        tensor = float("nan")
        if hm:
            tensor = 100.0 * to_float(r[ci[hm[0]]]) / 4.0 / g("smsp__cycles_elapsed.avg")
        table.append({"kernel": short(r[ci["Kernel Name"]]), "us": t_us, "grid": r[ci["launch__grid_size"]],
                      "regs": r[ci["launch__registers_per_thread"]], "tensor_busy_pct": tensor,
                      "issue_active_pct": g("smsp__issue_active.avg.pct_of_peak_sustained_active"),
                      "warps_active_pct": g("sm__warps_active.avg.pct_of_peak_sustained_active"),
                      "warp_inst_M": g("smsp__inst_executed.sum") / 1e6, "dram_read_MB": dr / 1e6, "dram_write_MB": dw / 1e6,
                      "dram_GBs": (dr + dw) / (t_us * 1e-6) / 1e9 if t_us > 0 else float("nan"),
                      "l2_hit_pct": g("lts__t_sector_hit_rate.pct")})
    return table


def md_table(table):
    out = ["| kernel | time (us) | grid | regs | tensor busy (% of cycles) | issue active (%) | warps active (%) | warp instr (M) | dram read (MB) | dram write (MB) | achieved dram GB/s | L2 hit (%) |",
           "|---|---|---|---|---|---|---|---|---|---|---|---|"]
    for r in table:
        out.append("| %s | %.1f | %s | %s | %.1f | %.1f | %.1f | %.2f | %.1f | %.1f | %.0f | %.1f |" % (
            r["kernel"], r["us"], r["grid"], r["regs"], r["tensor_busy_pct"], r["issue_active_pct"], r["warps_active_pct"],
            r["warp_inst_M"], r["dram_read_MB"], r["dram_write_MB"], r["dram_GBs"], r["l2_hit_pct"]))
    return "\n".join(out)


def launches(path):
    rows = [r for r in csv.reader(open(path)) if len(r) > 5]
    h = rows[0]
    ki, vi = h.index("Kernel Name"), h.index("Metric Value")
    lines = [(short(r[ki]), to_float(r[vi]) / 1e3) for r in rows[1:]]
    tot = sum(t for k, t in lines if "at::" not in k)
    out = ["| kernel | ncu time (us) | share of the library's kernels |", "|---|---|---|"]
    for k, t in lines:
        out.append("| %s | %.1f | %s |" % (k[:60], t, "-" if "at::" in k else "%.1f %%" % (100 * t / tot)))
    return "\n".join(out)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report", nargs="?")
    ap.add_argument("--launches")
    ap.add_argument("--md")
    ap.add_argument("--traffic")
    a = ap.parse_args()
    text = []
    if a.launches:
        text.append(launches(a.launches))
    if a.report:
        table = summarise(a.report)
        text.append(md_table(table))
        if a.traffic:
            acc = {}
            for r in table:
                acc.setdefault(r["kernel"], []).append((r["dram_read_MB"] + r["dram_write_MB"]) * 1e6)
            json.dump({k: int(sum(v) / len(v)) for k, v in acc.items()}, open(a.traffic, "w"), indent=1)
    s = "\n\n".join(text) + "\n"
    if a.md:
        open(a.md, "a").write(s)
    sys.stdout.write(s)


if __name__ == "__main__":
    main()
