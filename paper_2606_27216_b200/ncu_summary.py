"""Turn an Nsight Compute report (.ncu-rep) into the markdown tables kept under profiles/.

    python -m paper_2606_27216_b200.ncu_summary <report.ncu-rep> [--title "..."] [--command "..."] > profiles/<name>.md
    python -m paper_2606_27216_b200.ncu_summary <report.ncu-rep> --traffic T=128 [T=...]    # one CSV row per launch

Reads `ncu -i <report> --page raw --csv` (ncu is on the image; no GPU needed) and keeps the metrics the roofline
discussion uses: duration, clocks, registers, shared memory, tensor-pipe and issue utilisation, DRAM bytes and
bandwidth, shared-memory wavefronts, TMEM instruction counts, the warp-stall reasons.  Development tooling: nothing in
the library or the tests imports it.
"""
from __future__ import annotations

import csv
import io
import subprocess
import sys

KEEP = [
    "gpu__time_duration.sum",
    "sm__cycles_elapsed.avg",
    "sm__cycles_elapsed.avg.per_second",
    "launch__grid_size",
    "launch__block_size",
    "launch__registers_per_thread",
    "launch__shared_mem_per_block_dynamic",
    "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_elapsed",
    "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_tensor_subpipe_hmma.avg.pct_of_peak_sustained_active",
    "dram__bytes_read.sum",
    "dram__bytes_write.sum",
    "dram__bytes_read.sum.per_second",
    "dram__bytes_write.sum.per_second",
    "dram__throughput.avg.pct_of_peak_sustained_elapsed",
    "sm__throughput.avg.pct_of_peak_sustained_elapsed",
    "sm__issue_active.avg.pct_of_peak_sustained_elapsed",
    "smsp__inst_executed.sum",
    "sm__warps_active.avg.per_cycle_active",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed",
    "l1tex__data_pipe_tc_wavefronts_mem_shared.sum",
    "l1tex__data_pipe_tc_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "l1tex__t_sectors_pipe_lsu_mem_local_op_ld.sum",
    "l1tex__t_sectors_pipe_lsu_mem_local_op_st.sum",
    "smsp__sass_inst_executed_op_tmem_ldt.sum",
    "smsp__sass_inst_executed_op_tmem_stt.sum",
    "lts__t_sector_hit_rate.pct",
    "lts__throughput.avg.pct_of_peak_sustained_elapsed",
]
STALL_PREFIX = "smsp__average_warps_issue_stalled_"
STALL_SUFFIX = "_per_issue_active.ratio"


def raw_rows(report: str):
    out = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    hdr, units = rows[0], rows[1]
    return hdr, units, rows[2:]


def main(argv):
    if not argv:
        sys.exit(__doc__)
    report = argv[0]
    title = argv[argv.index("--title") + 1] if "--title" in argv else f"ncu --set full: {report}"
    command = argv[argv.index("--command") + 1] if "--command" in argv else None
    hdr, units, launches = raw_rows(report)
    col = {h: i for i, h in enumerate(hdr)}
    if "--traffic" in argv:
        tags = argv[argv.index("--traffic") + 1:]
        for li, r in enumerate(launches):
            def val(name):
                v, u = float(r[col[name]]), units[col[name]]
                return v * {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(u, 1.0)
            rd, wr = val("dram__bytes_read.sum"), val("dram__bytes_write.sum")
            name = r[col["Kernel Name"]].split("(")[0].split("::")[-1]
            print(f"{name},{tags[li] if li < len(tags) else ''},{rd:.0f},{wr:.0f}")
        return
    print(f"# {title}\n")
    if command:
        print("Command (run under gpurun on one B200):\n")
        print(f"    {command}\n")
    print("Table written by `python -m paper_2606_27216_b200.ncu_summary <report>` from `ncu -i <report> --page raw --csv`.\n")
    for li, r in enumerate(launches):
        name = r[col["Kernel Name"]][:90] if "Kernel Name" in col else "?"
        grid = r[col["Grid Size"]] if "Grid Size" in col else "?"
        block = r[col["Block Size"]] if "Block Size" in col else "?"
        print(f"## launch {li}: {name}  grid {grid} block {block}\n")
        print("| metric | unit | value |\n|---|---|---|")
        for k in KEEP:
            if k in col:
                print(f"| {k} | {units[col[k]]} | {r[col[k]]} |")
        stalls = []
        for h, i in col.items():
            if h.startswith(STALL_PREFIX) and h.endswith(STALL_SUFFIX):
                try:
                    stalls.append((float(r[i]), h[len(STALL_PREFIX):-len(STALL_SUFFIX)]))
                except ValueError:
                    pass
        for v, n in sorted(stalls, reverse=True)[:8]:
            print(f"| stall: {n} (warps per issue) | | {v:.3f} |")
        print()


if __name__ == "__main__":
    main(sys.argv[1:])
