"""Summarise an Nsight Compute raw page as the per-launch CSV that profiles/ keeps and bench.py reads.

    ncu -i capture.ncu-rep --page raw --csv > raw.csv
    python -m paper_2606_13283_b200.ncu_summary raw.csv > profiles/<name>_ncu_full.csv

One row per profiled launch: the bench.py kernel class of the launch (empty when the kernel belongs to none), the
kernel name, its duration and DRAM bytes in plain units, and the occupancy / pipe / stall columns the profile notes
quote.  No arithmetic of the method lives here: it only renames, converts units and selects columns.
"""
from __future__ import annotations

import csv
import re
import sys

# kernel-name pattern -> bench.py / arche_profile_get class
CLASSES = [
    (r"pointwise_g_kernel<.*LoadPotentialG", "potential_g"),
    (r"pointwise_g_kernel<.*StoreNhatA", "reduce_g"),
    (r"s5_rows_kernel", "reduce_g"),
    (r"pointwise_r_kernel<.*StoreVi", "vi_r"),
    (r"pointwise_r_kernel<.*LoadDensity", "density_r"),
    (r"mu_solve_kernel", "mu_pass"),
    (r"fft_yz\w*kernel<\d+, 2, (1|true)", "fft_inv_z_potential"),
    (r"fft_yz\w*kernel<\d+, 2, (0|false)", "fft_fwd_z_reduce"),
    (r"fft_yz\w*kernel<\d+, 1,", "fft_y"),
    (r"fft_c2r\w*kernel", "fft_inv_x_vi"),
    (r"fft_r2c\w*kernel", "fft_fwd_x_real"),
    (r"structure_factor", "structure_factor"),
    (r"force_kernel", "force"),
    (r"force_cols_kernel|force_w_kernel", "force"),
    (r"stress_fields_kernel", "stress_fields"),
    (r"scf_persistent_kernel", "scf_persistent"),
]
UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
        "ns": 1e-3, "us": 1.0, "usecond": 1.0, "ms": 1e3, "msecond": 1e3, "nsecond": 1e-3, "second": 1e6, "s": 1e6}
KEEP = [("gpu__time_duration.sum", "time_us"), ("dram__bytes_read.sum", "dram_bytes_read"),
        ("dram__bytes_write.sum", "dram_bytes_write"), ("lts__t_sector_hit_rate.pct", "l2_hit_pct"),
        ("sm__warps_active.avg.pct_of_peak_sustained_active", "warps_active_pct"),
        ("launch__registers_per_thread", "registers"), ("launch__grid_size", "grid"), ("launch__block_size", "block"),
        ("sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active", "fp64_pipe_pct"),
        ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue_active_pct"),
        ("l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed", "lsu_wavefronts_pct"),
        ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "smem_bank_conflicts"),
        ("dram__throughput.avg.pct_of_peak_sustained_elapsed", "dram_throughput_pct"),
        ("smsp__inst_executed.sum", "instructions")]
STALL = re.compile(r"smsp__average_warps_issue_stalled_(\w+)_per_issue_active\.ratio")


def classify(name: str) -> str:
    for pat, cls in CLASSES:
        if re.search(pat, name):
            return cls
    return ""


def num(v: str) -> float:
    try:
        return float(v.replace(",", ""))
    except ValueError:
        return float("nan")


def summarise(rows):
    head, units, data = rows[0], rows[1], rows[2:]
    col = {h: i for i, h in enumerate(head)}
    stall_cols = [(STALL.match(h).group(1), i) for i, h in enumerate(head) if STALL.match(h)]
    out = [["class", "kernel"] + [k for _, k in KEEP] + ["top_stalls_warps_per_issue"]]
    for r in data:
        name = r[col["Kernel Name"]]
        line = [classify(name), name]
        for metric, _ in KEEP:
            if metric not in col:
                line.append("")
                continue
            v = num(r[col[metric]]) * UNIT.get(units[col[metric]], 1.0)
            line.append(f"{v:.6g}")
        st = sorted(((num(r[i]), s) for s, i in stall_cols if num(r[i]) == num(r[i])), reverse=True)[:4]
        line.append("; ".join(f"{s} {v:.2f}" for v, s in st))
        out.append(line)
    return out


def main(argv):
    src = open(argv[1], newline="") if len(argv) > 1 else sys.stdin
    rows = [r for r in csv.reader(src) if r and (r[0] == "ID" or r[0].isdigit() or r[0] == "")]
    w = csv.writer(sys.stdout)
    for line in summarise(rows):
        w.writerow(line)


if __name__ == "__main__":
    main(sys.argv)
