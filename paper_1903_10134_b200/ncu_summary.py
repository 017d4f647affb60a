"""Turns `ncu -i <report> --page raw --csv` output into the summary bench.py reads for `roofline.traffic`.

    python -m paper_1903_10134_b200.ncu_summary raw.csv --workload 4a --commit <hash> --command "<the ncu command>"

writes profiles/ncu_r2_<workload>.json (per kernel: launches averaged, duration, DRAM bytes per launch, warp
instructions, issue-slot and pipe utilisation, shared-memory wavefronts and bank-conflict wavefronts, occupancy) together
with the SHA-256 of csrc/mdpd_b200.cu, so that bench.py can tell a capture of another build from a current one, and
prints the same numbers as a markdown table.  Launches of the rebuild chain that returned at once (the trigger did not
fire) are left out: only launches longer than 20 % of the kernel's longest launch count.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import json
import os
import re

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
SRC = os.path.join(PKG, "csrc", "mdpd_b200.cu")

UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
        "ns": 1e-6, "us": 1e-3, "ms": 1.0, "s": 1e3, "ns ": 1e-6}

METRICS = {
    "ms": "gpu__time_duration.sum",
    "dram_read": "dram__bytes_read.sum",
    "dram_write": "dram__bytes_write.sum",
    "warp_inst": "smsp__inst_executed.sum",
    "issue_active_pct": "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "warps_per_sm": "sm__warps_active.avg.per_cycle_active",
    "threads_per_inst": "smsp__thread_inst_executed_per_inst_executed.ratio",
    "smem_wavefronts": "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum",
    "smem_conflict_wavefronts": "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "smem_pipe_pct": "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed",
    "l1_pipe_pct": "l1tex__data_pipe_lsu_wavefronts.sum.pct_of_peak_sustained_elapsed",
    "stall_long_scoreboard": "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio",
    "stall_short_scoreboard": "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio",
    "stall_barrier": "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio",
    "stall_wait": "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio",
    "stall_not_selected": "smsp__average_warps_issue_stalled_not_selected_per_issue_active.ratio",
    "stall_math_pipe": "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio",
    "stall_mio": "smsp__average_warps_issue_stalled_mio_throttle_per_issue_active.ratio",
    "pipe_alu_pct": "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
    "pipe_fma_pct": "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
    "pipe_xu_pct": "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
    "pipe_lsu_pct": "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
    "registers": "launch__registers_per_thread",
    "block": "launch__block_size",
    "grid": "launch__grid_size",
    "l2_hit_pct": "lts__t_sector_hit_rate.pct",
}


def kernel_key(name: str) -> str:
    m = re.search(r"(k_[a-z_]+)(<([^>]*)>)?", name)
    if not m:
        return name
    base = m.group(1)
    if base == "k_cells":
        mode = (m.group(3) or "0").split(",")[0].strip()
        return "k_cells_list" if mode == "0" else "k_cells_direct"
    return base


def summarise(path: str):
    rows = list(csv.reader(open(path)))
    hdr, units = rows[0], rows[1]
    col = {h: i for i, h in enumerate(hdr)}
    per = {}
    for r in rows[2:]:
        if len(r) != len(hdr):
            continue
        key = kernel_key(r[col["Kernel Name"]])
        ent = {}
        for short, metric in METRICS.items():
            if metric not in col:
                continue
            try:
                v = float(r[col[metric]])
            except ValueError:
                continue
            ent[short] = v * UNIT.get(units[col[metric]].strip(), 1.0)
        per.setdefault(key, []).append(ent)
    out = {}
    for key, launches in per.items():
        longest = max(e.get("ms", 0.0) for e in launches)
        real = [e for e in launches if e.get("ms", 0.0) > 0.2 * longest]
        avg = {k: sum(e[k] for e in real if k in e) / max(1, sum(1 for e in real if k in e)) for k in METRICS if any(k in e for e in real)}
        ent = {"launches_averaged": len(real), "launches_captured": len(launches), "gpu_time_ms": round(avg.get("ms", 0.0), 5),
               "dram_bytes_per_launch": round(avg.get("dram_read", 0.0) + avg.get("dram_write", 0.0)),
               "dram_read_bytes": round(avg.get("dram_read", 0.0)), "dram_write_bytes": round(avg.get("dram_write", 0.0)),
               "smem_pipe_frac": round(avg.get("smem_pipe_pct", 0.0) / 100.0, 4),
               "l1_data_pipe_frac": round(avg.get("l1_pipe_pct", 0.0) / 100.0, 4),
               # warps of a scheduler waiting for each reason, per cycle in which the scheduler issued
               "stalls_per_issue": {k[6:]: round(avg[k], 3) for k in METRICS if k.startswith("stall_") and k in avg}}
        for k in ("warp_inst", "issue_active_pct", "warps_per_sm", "threads_per_inst", "smem_wavefronts",
                  "smem_conflict_wavefronts", "pipe_alu_pct", "pipe_fma_pct", "pipe_xu_pct", "pipe_lsu_pct", "registers",
                  "block", "grid", "l2_hit_pct"):
            if k in avg:
                ent[k] = round(avg[k], 3)
        out[key] = ent
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--workload", required=True)
    ap.add_argument("--commit", required=True)
    ap.add_argument("--command", required=True)
    ap.add_argument("--particles", type=int, default=0)
    a = ap.parse_args()
    kernels = summarise(a.raw_csv)
    doc = {"workload": a.workload, "commit": a.commit, "command": a.command,
           "kernel_source_sha256": hashlib.sha256(open(SRC, "rb").read()).hexdigest(),
           "note": "ncu --set full replays every kernel ~40 times with cold caches and serialised launches: durations are a "
                   "few % above the CUDA-event times of a plain run; a number printed under ncu is never a bench value",
           "kernels": kernels}
    dst = os.path.join(ROOT, "profiles", f"ncu_r2_{a.workload}.json")
    json.dump(doc, open(dst, "w"), indent=1)
    n = a.particles
    print(f"| kernel | launches | ms | DRAM MB (r + w) | {'B/particle | ' if n else ''}warp inst{'/particle' if n else ''} | issue % | L1 data pipe % (shared part) | "
          "conflict / all wavefronts | alu / fma / xu / lsu pipe % | warps/SM | regs x block | stalled warps per issue: long sb / short sb / barrier / wait |")
    print("|---|---:|---:|---:|" + ("---:|" if n else "") + "---:|---:|---:|---:|---:|---:|---:|---:|")
    for k, e in sorted(kernels.items(), key=lambda kv: -kv[1]["gpu_time_ms"]):
        wi = e.get("warp_inst", 0.0)
        cells = [k, f"{e['launches_averaged']} of {e['launches_captured']}", f"{e['gpu_time_ms']:.4f}",
                 f"{e['dram_read_bytes'] / 1e6:.1f} + {e['dram_write_bytes'] / 1e6:.1f}"]
        if n:
            cells.append(f"{e['dram_bytes_per_launch'] / n:.1f}")
        cells += [f"{wi / n:.1f}" if n else f"{wi:.3g}", f"{e.get('issue_active_pct', 0):.1f}",
                  f"{100 * e['l1_data_pipe_frac']:.1f} ({100 * e['smem_pipe_frac']:.1f})",
                  f"{e.get('smem_conflict_wavefronts', 0):.3g} / {e.get('smem_wavefronts', 0):.3g}",
                  f"{e.get('pipe_alu_pct', 0):.0f} / {e.get('pipe_fma_pct', 0):.0f} / {e.get('pipe_xu_pct', 0):.0f} / {e.get('pipe_lsu_pct', 0):.0f}",
                  f"{e.get('warps_per_sm', 0):.1f}", f"{e.get('registers', 0):.0f} x {e.get('block', 0):.0f}",
                  " / ".join(f"{e['stalls_per_issue'].get(q, 0):.2f}" for q in ("long_scoreboard", "short_scoreboard", "barrier", "wait"))]
        print("| " + " | ".join(cells) + " |")
    print(f"\nwritten: {dst}")


if __name__ == "__main__":
    main()
