"""Turn an `ncu --set full` report of one step (ncu_step.py) into the per-kernel CSV that bench.py's
`roofline.traffic` reads and the tables under profiles/ are built from.  Runs where ncu is installed
(no GPU needed):

  python -m paper_2505_22313_b200.ncu_summary gpurun_out/prof_C5.ncu-rep gpurun_out/labels_C5.json \
         profiles/r02_ncu_C5.csv

One row per launch of the profiled step, in launch order: pass label (from ncu_step.py), kernel name,
device time, DRAM bytes read / written, and the utilisation and stall figures quoted in DESIGN.md.
The first line records the hash of the kernel sources the capture is valid for."""
from __future__ import annotations

import csv
import io
import json
import subprocess
import sys

from . import build as dop_build

METRICS = [
    ("time_us", "gpu__time_duration.sum"),
    ("dram_bytes_read", "dram__bytes_read.sum"),
    ("dram_bytes_write", "dram__bytes_write.sum"),
    ("dram_pct", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed"),
    ("issue_active_pct", "smsp__issue_active.avg.pct_of_peak_sustained_active"),
    ("warps_active_pct", "sm__warps_active.avg.pct_of_peak_sustained_active"),
    ("l1_wavefronts_pct", "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed"),
    ("smem_wavefronts", "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum"),
    ("smem_bank_conflicts", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum"),
    ("inst_executed", "smsp__inst_executed.sum"),
    ("registers", "launch__registers_per_thread"),
    ("stall_long_scoreboard", "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio"),
    ("stall_mio_throttle", "smsp__average_warps_issue_stalled_mio_throttle_per_issue_active.ratio"),
    ("stall_lg_throttle", "smsp__average_warps_issue_stalled_lg_throttle_per_issue_active.ratio"),
    ("stall_barrier", "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio"),
    ("stall_short_scoreboard", "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio"),
    ("stall_math_throttle", "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio"),
    ("stall_wait", "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio"),
]
UNIT_SCALE = {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12, "byte": 1.0,
              "ns": 1e-3, "us": 1.0, "usecond": 1.0, "ms": 1e3, "msecond": 1e3, "nsecond": 1e-3, "second": 1e6, "s": 1e6}


def main() -> None:
    rep, labels_path, out_path = sys.argv[1:4]
    with open(labels_path) as f:
        meta = json.load(f)
    raw = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(raw)))
    hdr, units, data = rows[0], rows[1], rows[2:]
    if len(data) != len(meta["labels"]):
        raise SystemExit(f"{len(data)} captured launches but {len(meta['labels'])} pass labels: not one whole step")
    kcol = hdr.index("Kernel Name")
    with open(out_path, "w", newline="") as f:
        f.write(f"# source_stamp={dop_build.source_stamp()}\n")
        f.write(f"# config={meta['config']} points_per_plane={meta['points_per_plane']} "
                f"(ncu --set full, one forward+adjoint step, launch order; bytes are per launch)\n")
        w = csv.writer(f)
        w.writerow(["pass", "kernel"] + [m for m, _ in METRICS])
        for label, r in zip(meta["labels"], data):
            out = [label, r[kcol]]
            for short, name in METRICS:
                if name not in hdr:
                    out.append("")
                    continue
                i = hdr.index(name)
                v = float(r[i].replace(",", "")) if r[i] not in ("", "n/a") else float("nan")
                v *= UNIT_SCALE.get(units[i], 1.0) if short in ("time_us", "dram_bytes_read", "dram_bytes_write") else 1.0
                out.append(f"{v:.6g}")
            w.writerow(out)
    print(out_path)


if __name__ == "__main__":
    main()
