"""Summarise an `ncu --set full` capture of one bench step as text: one table row per kernel launch, and the DRAM
traffic per C-ABI call that bench.py prints as `roofline.traffic`.

    ncu -i capture.ncu-rep --page raw --csv > raw.csv
    python -m paper_2412_20522_b200.ncu_summary raw.csv --config 3 --md profiles/r02_ncu_table.md \
        --traffic-json profiles/r02_traffic.json

Reads the CSV only (no GPU, no ncu needed here).  Kernels are attributed to the call of include/mg.h that launches them.
"""
import argparse
import csv
import json
import os

COLS = [("Kernel Name", "kernel"), ("gpu__time_duration.sum", "time"), ("dram__bytes_read.sum", "dram_rd"),
        ("dram__bytes_write.sum", "dram_wr"), ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "dram%"),
        ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue%"), ("smsp__inst_executed.sum", "warp_inst"),
        ("smsp__thread_inst_executed_per_inst_executed.ratio", "act_thr"),
        ("sm__warps_active.avg.pct_of_peak_sustained_active", "warps_act%"), ("launch__registers_per_thread", "regs"),
        ("sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active", "fma%"),
        ("sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "alu%"),
        ("sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active", "xu%"),
        ("lts__throughput.avg.pct_of_peak_sustained_elapsed", "lts%"),
        ("l1tex__throughput.avg.pct_of_peak_sustained_elapsed", "l1tex%")]

CALL_OF = [("preprocess_bwd", "preprocess_bwd"), ("preprocess_kernel", "preprocess"), ("render_fwd", "render_fwd"),
           ("render_bwd", "render_bwd"), ("depth_keys", "bin_sort"), ("depth_hist", "bin_sort"), ("ctl_", "bin_sort"), ("radix_", "bin_sort"),
           ("row_expand", "bin_sort"), ("col_expand", "bin_sort"), ("scan_", "bin_sort"), ("plan_", "bin_sort"),
           ("tile_ranges", "bin_sort"), ("tile_order", "bin_sort"), ("visible_", "bin_sort"), ("sort_", "bin_sort")]

UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "ns": 1e-3, "us": 1.0, "usecond": 1.0, "ms": 1e3,
              "msecond": 1e3, "nsecond": 1e-3}


def call_of(kernel):
    for key, call in CALL_OF:
        if key in kernel:
            return call
    return None


def short(name):
    return name.replace("<unnamed>::", "").replace("void ", "").split("(")[0][:40]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--md")
    ap.add_argument("--traffic-json")
    a = ap.parse_args()
    rows = list(csv.reader(open(a.raw_csv)))
    while rows and (not rows[0] or rows[0][0] != "ID"):  # ncu log lines before the header
        rows.pop(0)
    hdr, units, body = rows[0], rows[1], rows[2:]
    keep = [(hdr.index(c), n) for c, n in COLS if c in hdr]
    lines = ["| " + " | ".join(n for _, n in keep) + " |", "|" + "---|" * len(keep),
             "| " + " | ".join(units[i] for i, _ in keep) + " |"]
    traffic, time_us = {}, {}
    i_rd, i_wr, i_t, i_k = (hdr.index(c) for c in ("dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__time_duration.sum", "Kernel Name"))
    for r in body:
        if len(r) != len(hdr):
            continue
        cells = []
        for i, n in keep:
            try:
                cells.append(f"{float(r[i].replace(',', '')):.4g}")
            except ValueError:
                cells.append(short(r[i]))
        lines.append("| " + " | ".join(cells) + " |")
        call = call_of(r[i_k])
        if call:
            b = (float(r[i_rd].replace(",", "")) * UNIT_SCALE[units[i_rd]] + float(r[i_wr].replace(",", "")) * UNIT_SCALE[units[i_wr]])
            traffic[call] = traffic.get(call, 0.0) + b
            time_us[call] = time_us.get(call, 0.0) + float(r[i_t].replace(",", "")) * UNIT_SCALE[units[i_t]]
    lines += ["", "Per call (sum over its kernels; time under ncu is cold-cache and serialised):", "",
              "| call | kernels' time (us) | dram read + write (MB) |", "|---|---|---|"]
    for c in ("preprocess", "bin_sort", "render_fwd", "render_bwd", "preprocess_bwd"):
        if c in traffic:
            lines.append(f"| {c} | {time_us[c]:.1f} | {traffic[c] / 1e6:.1f} |")
    text = "\n".join(lines) + "\n"
    if a.md:
        open(a.md, "w").write(text)
    else:
        print(text)
    if a.traffic_json:
        data = json.load(open(a.traffic_json)) if os.path.exists(a.traffic_json) else {}
        data[str(a.config)] = {k: round(v) for k, v in traffic.items()}
        json.dump(data, open(a.traffic_json, "w"), indent=1, sort_keys=True)


if __name__ == "__main__":
    main()
