"""Summarise an `ncu --set full` capture of one bench step as text: one table row per kernel launch, and the DRAM
traffic per C-ABI call that bench.py prints as `roofline.traffic`.

    ncu -i capture.ncu-rep --page raw --csv > raw.csv
    python ncu_summary.py raw.csv --config 3 --md profiles/r03_ncu_table.md --traffic-json profiles/r03_traffic.json

Reads the CSV only (no GPU, no ncu needed here).  Kernels are attributed to the call of include/mg.h that launches them.
Measurement tooling: it lives beside bench.py, not in the product package.

Two tables, one row per kernel launch each.  The first is the compute view (time, DRAM bytes, issue and pipe
utilisation); the second is what north_star asks for on top of it -- shared-memory and L1 data-pipe utilisation against
peak and bank conflicts for the blend kernels, the `red` (atomic gradient scatter) instruction and sector counts, L1 / L2
hit rates, and the four largest warp-stall reasons per issued instruction.
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

# second table: memory pipes, atomics, hit rates (the stall reasons are picked per kernel, see stalls())
COLS2 = [("Kernel Name", "kernel"),
         ("l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed", "lsu_data_pipe%"),
         ("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed", "smem_wavefronts%"),
         ("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "smem_wavefronts"),
         ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "smem_bank_conflicts"),
         ("smsp__inst_executed_op_global_red.sum", "red_inst"),
         ("l1tex__t_sectors_pipe_lsu_mem_global_op_red.sum", "red_sectors"),
         ("lts__d_atomic_input_cycles_active.avg.pct_of_peak_sustained_elapsed", "l2_atomic_unit%"),
         ("l1tex__t_sector_hit_rate.pct", "l1_hit%"), ("lts__t_sector_hit_rate.pct", "l2_hit%")]
STALL_PREFIX, STALL_SUFFIX = "smsp__average_warps_issue_stalled_", "_per_issue_active.ratio"

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


def num(cell):
    return float(cell.replace(",", ""))


def stalls(hdr, r, top=4):
    """The `top` largest stall reasons of a launch as 'reason value' (warps stalled per issued instruction); `selected`
    (the warp that did issue) is not a stall and is left out."""
    out = []
    for i, h in enumerate(hdr):
        if h.startswith(STALL_PREFIX) and h.endswith(STALL_SUFFIX) and "not_issued" not in h:
            name = h[len(STALL_PREFIX):-len(STALL_SUFFIX)]
            if name != "selected":
                try:
                    out.append((num(r[i]), name))
                except ValueError:
                    pass
    return ", ".join(f"{n} {v:.2f}" for v, n in sorted(out, reverse=True)[:top])


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
    keep2 = [(hdr.index(c), n) for c, n in COLS2 if c in hdr]
    lines += ["", "Memory pipes, atomics, hit rates and the four largest stall reasons (warps stalled per issued instruction):", "",
              "| " + " | ".join(n for _, n in keep2) + " | stalls |", "|" + "---|" * (len(keep2) + 1)]
    for r in body:
        if len(r) != len(hdr):
            continue
        cells = []
        for i, n in keep2:
            try:
                cells.append(f"{num(r[i]):.4g}")
            except ValueError:
                cells.append(short(r[i]))
        lines.append("| " + " | ".join(cells) + " | " + stalls(hdr, r) + " |")
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
