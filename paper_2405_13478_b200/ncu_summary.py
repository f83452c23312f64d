"""Text summary of one kernel of an Nsight Compute report, for profiles/ (bench.py reads the DRAM
traffic of its `roofline.traffic` from such a file).

    python -m paper_2405_13478_b200.ncu_summary REPORT.ncu-rep [KERNEL_SUBSTRING [SNAPSHOTS_IN_LAUNCH]] > profiles/NAME_summary.txt

Runs `ncu -i REPORT --page raw --csv`, takes the LAST launch whose kernel name contains the substring
(default: the last launch in the report) and prints `metric  value  unit` lines for the metrics a
roofline argument needs, then the warp-stall reasons sorted by weight.  Two comment lines go in front for
bench.py: `# kernel_sources_sha16` (hash of csrc/ at capture time: bench.py flags a summary older than the
kernels) and, when given, `# snapshots_in_launch` (a capture of ONE launch pair of a chunked route, to be scaled
to the step).  A development tool, kept here because the files under profiles/ name it as their command."""
from __future__ import annotations

import csv
import subprocess
import sys

WANT = ["gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum",
        "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "dram__throughput.avg.pct_of_peak_sustained_elapsed",
        "sm__throughput.avg.pct_of_peak_sustained_elapsed", "smsp__inst_executed.sum",
        "sm__inst_executed.avg.per_cycle_elapsed", "sm__inst_executed.avg.per_cycle_active",
        "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__warps_active.avg.pct_of_peak_sustained_active",
        "launch__registers_per_thread", "launch__grid_size", "launch__block_size",
        "launch__shared_mem_per_block_dynamic", "launch__occupancy_limit_registers",
        "launch__occupancy_limit_shared_mem", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
        "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "lts__t_sector_hit_rate.pct",
        "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
        "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active",
        "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active",
        "sm__inst_executed_pipe_tensor.sum", "lts__throughput.avg.pct_of_peak_sustained_elapsed"]


def main(argv):
    if len(argv) < 2:
        raise SystemExit(__doc__)
    rep, sub = argv[1], (argv[2] if len(argv) > 2 else "")
    out = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(out.splitlines()))
    head, units, data = rows[0], rows[1], rows[2:]
    kcol = head.index("Kernel Name")
    pick = [r for r in data if sub in r[kcol]]
    if not pick:
        raise SystemExit(f"no launch matching {sub!r}")
    r = pick[-1]
    print(f"# {r[kcol]}  (launch {len(pick)} of {len(pick)} matching {sub!r}; report {rep})")
    import os
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    from bench import kernel_sources_sha16
    print(f"# kernel_sources_sha16 {kernel_sources_sha16()}")
    if len(argv) > 3:
        print(f"# snapshots_in_launch {int(argv[3])}")
    for name in WANT:
        if name in head:
            i = head.index(name)
            print(f"{name:<80} {r[i]} {units[i]}")
    stalls = []
    for i, name in enumerate(head):
        if "average_warps_issue_stalled" in name and name.endswith("per_issue_active.ratio"):
            try:
                stalls.append((float(r[i].replace(",", "")), name))
            except ValueError:
                pass
    for v, name in sorted(stalls, reverse=True):
        print(f"  {name:<88} {v:.6f}")


if __name__ == "__main__":
    main(sys.argv)
