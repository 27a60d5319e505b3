"""Text summary of an `ncu --set full` capture of the bfsc kernels (the files under profiles/ that bench.py reads).

    ncu -i capture.ncu-rep --page raw --csv > capture.csv
    python -m paper_1704_00513_b200.ncu_summary capture.csv --kernel k_enc_tiles --labels a,b,c > summary.txt

The capture is made with `bench.py --ncu` (profiles/README.md has the full command): between cudaProfilerStart and
cudaProfilerStop it runs, for each of the streams a, b, c of BASELINE.json configs[1] in this order, ONE compress call
and ONE decompress call, so the n-th launch of a kernel in the capture belongs to the n-th label. Output: one
`== stream <label>` section per launch with `metric value` lines, units as ncu prints them. No arithmetic of the
codec here; reading a csv only.
"""
from __future__ import annotations

import argparse
import csv
import sys

METRICS = [
    "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "smsp__inst_executed.sum",
    "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__warps_active.avg.pct_of_peak_sustained_active",
    "launch__registers_per_thread", "launch__grid_size", "launch__block_size", "launch__occupancy_limit_registers",
    "launch__occupancy_limit_shared_mem", "launch__occupancy_limit_warps", "lts__t_sector_hit_rate.pct",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum",
    "sm__cycles_elapsed.avg.per_second", "smsp__cycles_active.avg",
    "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
    "l1tex__t_requests_pipe_lsu_mem_global_op_ld.sum", "l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum",
    "l1tex__t_requests_pipe_lsu_mem_global_op_st.sum", "l1tex__t_sectors_pipe_lsu_mem_global_op_st.sum",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
]
# bench.py reads the time in us and the DRAM bytes in MB: normalised here whatever unit ncu chose for the column
TO_US = {"nsecond": 1e-3, "usecond": 1.0, "msecond": 1e3, "second": 1e6}
TO_MB = {"byte": 1e-6, "Kbyte": 1e-3, "Mbyte": 1.0, "Gbyte": 1e3}
STALL_PREFIX, STALL_SUFFIX = "smsp__average_warps_issue_stalled_", "_per_issue_active.ratio"


def rows_of(path):
    """(header, unit row, data rows) of an `ncu --page raw --csv` file; lines before the header (ncu's ==PROF== chatter
    when the csv was written with --log-file) are skipped."""
    with open(path, newline="") as f:
        rows = list(csv.reader(f))
    for i, r in enumerate(rows):
        if "Kernel Name" in r:
            return r, rows[i + 1], rows[i + 2:]
    raise SystemExit(f"{path}: no 'Kernel Name' column: not an ncu raw-page csv")


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("csv")
    ap.add_argument("--kernel", required=True, help="substring of the kernel name, e.g. k_enc_tiles")
    ap.add_argument("--labels", default="a,b,c", help="label of the 1st, 2nd, ... launch of that kernel")
    ap.add_argument("--title", default="")
    a = ap.parse_args(argv)
    header, units, data = rows_of(a.csv)
    col = {n: i for i, n in enumerate(header)}
    labels = a.labels.split(",")
    hits = [r for r in data if len(r) == len(header) and a.kernel in r[col["Kernel Name"]]]
    if a.title:
        print(a.title)
    print(f"source: {a.csv}; {len(hits)} launches of *{a.kernel}*; gpu__time_duration.sum in us, dram__bytes_* in MB, "
          "everything else in the unit ncu prints")
    for k, r in enumerate(hits):
        label = labels[k] if k < len(labels) else f"#{k}"
        print(f"\n== stream {label} : {r[col['Kernel Name']]}  grid {r[col['Grid Size']] if 'Grid Size' in col else '?'}")
        for m in METRICS:
            if m not in col:
                continue
            v, u = r[col[m]], units[col[m]]
            if m == "gpu__time_duration.sum" and u in TO_US:
                v = f"{float(v.replace(',', '')) * TO_US[u]:.3f}"
            elif m.startswith("dram__bytes_") and u in TO_MB:
                v = f"{float(v.replace(',', '')) * TO_MB[u]:.6f}"
            print(m, v)
        for n in header:
            if n.startswith(STALL_PREFIX) and n.endswith(STALL_SUFFIX) and "not_issued" not in n:
                print("stall_" + n[len(STALL_PREFIX):-len(STALL_SUFFIX)], r[col[n]])
    return 0


if __name__ == "__main__":
    sys.exit(main())
