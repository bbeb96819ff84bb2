"""Turns Nsight Compute reports of the hot kernels into the committed evidence under profiles/.

    python -m paper_1711_00975_b200.profile_capture --tag r2 --workload cfg3 --particles-per-launch 134217728 \
        --command "<the command the reports were captured with>" gpurun_out/a.ncu-rep [gpurun_out/b.ncu-rep ...]

For every kernel launch in the reports it writes profiles/<tag>_ncu_<kernel>.csv (a two-column `metric,value` export of
`ncu -i <rep> --page raw --csv`, the metrics that matter for the roofline plus every stall reason) and updates
profiles/<tag>_kernel_metrics.json, which bench.py reads for `roofline.traffic` and the instruction count per particle.
The json records the hash of the kernel sources it was captured on (bench.kernel_sources_sha); bench.py ignores it
once those sources change.  Needs `ncu` on PATH (reading a report needs no GPU).  Not imported by the library.

    python -m paper_1711_00975_b200.profile_capture --launch-list gpurun_out/r2_launches_cfg3.csv profiles/r2_launches_cfg3_last_step.csv

turns the launch list of `ncu --metrics gpu__time_duration.sum --csv --log-file <raw> ... bench.py` into the rows of the
last step and prints the per-kernel summary.
"""
from __future__ import annotations

import argparse
import csv
import json
import re
import subprocess
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))

KEEP = re.compile(
    r"^(gpu__time_duration\.sum|smsp__inst_executed\.sum|smsp__thread_inst_executed\.sum|smsp__issue_active\.avg\.pct_of_peak_sustained_active|"
    r"sm__warps_active\.avg\.pct_of_peak_sustained_active|sm__throughput\.avg\.pct_of_peak_sustained_elapsed|"
    r"sm__pipe_(alu|fma)_cycles_active\.avg\.pct_of_peak_sustained_active|sm__inst_executed_pipe_lsu\.avg\.pct_of_peak_sustained_active|"
    r"l1tex__throughput\.avg\.pct_of_peak_sustained_active|l1tex__data_pipe_lsu_wavefronts_mem_shared\.sum|"
    r"l1tex__data_bank_conflicts_pipe_lsu_mem_shared\.sum|lts__t_sectors\.sum|lts__t_sector_hit_rate\.pct|"
    r"lts__throughput\.avg\.pct_of_peak_sustained_elapsed|lts__t_sectors_op_(red|atom|read|write)\.sum|"
    r"dram__bytes_(read|write)\.sum|dram__throughput\.avg\.pct_of_peak_sustained_elapsed|gpu__dram_throughput\.avg\.pct_of_peak_sustained_elapsed|"
    r"launch__(registers_per_thread|grid_size|block_size|shared_mem_per_block_dynamic|occupancy_limit_\w+)|"
    r"smsp__average_warp_latency_per_inst_issued\.ratio|smsp__average_warps_issue_stalled_\w+_per_issue_active\.ratio)$")


def raw_rows(rep: Path):
    out = subprocess.run(["ncu", "-i", str(rep), "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(out.splitlines()))
    hdr, units = rows[0], rows[1]
    for r in rows[2:]:
        yield {h: (v, u) for h, u, v in zip(hdr, units, r)}


def short_name(full: str) -> str:
    m = re.search(r"(k_[a-z_0-9]+)\s*(<[^>]*>)?", full)
    name = m.group(1) + (m.group(2) or "") if m else full
    return re.sub(r"[^A-Za-z0-9_]+", "_", name).strip("_")


UPDATE_KERNELS = ("k_bin_scatter", "k_bin_apply", "k_update", "k_compact_kept")


def launch_list(raw_csv: Path, out_csv: Path):
    """`ncu --metrics gpu__time_duration.sum --csv --log-file raw_csv ... bench.py` -> the launches of the LAST step (a step
    starts where an update kernel follows a kernel of the scan / select phases), one row per launch, and a per-kernel
    summary (markdown) on stdout.  The probe kernels bench.py runs for its denominators are left out."""
    lines = [l for l in raw_csv.read_text().splitlines() if l.startswith('"')]
    rows = list(csv.DictReader(lines))
    seq = []
    for r in rows:
        if r["Metric Name"] != "gpu__time_duration.sum":
            continue
        name = re.sub(r"^void\s+", "", r["Kernel Name"])
        name = re.sub(r"\(.*$", "", name).replace("cs::", "").replace("(anonymous namespace)::", "")
        if name.startswith("k_probe"):
            continue
        ns = float(r["Metric Value"]) * {"ns": 1.0, "us": 1e3, "ms": 1e6, "s": 1e9}[r["Metric Unit"]]
        seq.append((name, ns))
    starts = [i for i, (nm, _) in enumerate(seq)
              if nm.startswith(UPDATE_KERNELS) and (i == 0 or not seq[i - 1][0].startswith(UPDATE_KERNELS))]
    last = seq[starts[-1]:] if starts else seq
    with open(out_csv, "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(["launch", "kernel", "gpu__time_duration.sum [ns]"])
        for i, (nm, ns) in enumerate(last):
            w.writerow([i, nm, int(round(ns))])
    agg = {}
    for nm, ns in last:
        c, t = agg.get(nm, (0, 0.0))
        agg[nm] = (c + 1, t + ns)
    total = sum(t for _, t in agg.values())
    print(f"steps found: {len(starts)}; last step: {len(last)} launches, {total / 1e6:.3f} ms under ncu\n")
    print("| Kernel | Launches | Total ms (ncu) | Share |\n|---|---|---|---|")
    for nm, (c, t) in sorted(agg.items(), key=lambda kv: -kv[1][1]):
        print(f"| `{nm}` | {c} | {t / 1e6:.3f} | {100 * t / total:.1f} % |")
    print(f"| sum | {len(last)} | {total / 1e6:.2f} | |")
    print("wrote", out_csv)


def main():
    if len(sys.argv) > 1 and sys.argv[1] == "--launch-list":
        launch_list(Path(sys.argv[2]), Path(sys.argv[3]))
        return
    ap = argparse.ArgumentParser()
    ap.add_argument("reports", nargs="+")
    ap.add_argument("--tag", default="r2")
    ap.add_argument("--workload", required=True)
    ap.add_argument("--particles-per-launch", type=int, required=True, help="particles one launch of the scatter kernel covers")
    ap.add_argument("--passes-per-particle", type=int, default=1, help="scatter launches that touch each kept particle")
    ap.add_argument("--command", required=True, help="the full command line the reports were captured with")
    a = ap.parse_args()
    import bench
    prof = ROOT / "profiles"
    meta_path = prof / f"{a.tag}_kernel_metrics.json"
    sha = bench.kernel_sources_sha()
    meta = {}
    if meta_path.exists():
        meta = json.loads(meta_path.read_text())
        if meta.get("kernel_sources_sha") != sha:
            meta = {}
    meta.setdefault("kernel_sources_sha", sha)
    meta.setdefault("kernel_sources", bench.KERNEL_SOURCES)
    meta.setdefault("workloads", {})
    meta["command"] = a.command
    wl = meta["workloads"].setdefault(a.workload, {})
    for rep in a.reports:
        for row in raw_rows(Path(rep)):
            full = row["Kernel Name"][0]
            name = short_name(full)
            path = prof / f"{a.tag}_ncu_{a.workload}_{name}.csv"
            with open(path, "w", newline="") as f:
                w = csv.writer(f)
                w.writerow(["metric", "value", "unit"])
                w.writerow(["kernel", full, ""])
                w.writerow(["captured_with", a.command, ""])
                w.writerow(["kernel_sources_sha", sha, ""])
                for h, (v, u) in row.items():
                    if KEEP.match(h):
                        w.writerow([h, v, u])
            def val(k, scale=1.0):
                v, u = row[k]
                v = float(v)
                mult = {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12, "byte": 1.0, "us": 1e-3, "ms": 1.0, "ns": 1e-6,
                        "s": 1e3}.get(u, 1.0)
                return v * mult * scale
            entry = {"dram_bytes_per_launch": val("dram__bytes_read.sum") + val("dram__bytes_write.sum"),
                     "duration_ms_under_ncu": val("gpu__time_duration.sum"),
                     "warp_instructions_per_launch": val("smsp__inst_executed.sum"),
                     "issue_active_pct": val("smsp__issue_active.avg.pct_of_peak_sustained_active"),
                     "alu_pipe_pct": val("sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active"),
                     "fma_pipe_pct": val("sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active"),
                     "source": path.name}
            key = re.match(r"k_[a-z_]+", name).group(0).rstrip("_")
            if key == "k_bin_scatter":
                entry["thread_instructions_per_particle"] = 32.0 * entry["warp_instructions_per_launch"] / a.particles_per_launch
                entry["passes_per_particle"] = a.passes_per_particle
                entry["particles_per_launch"] = a.particles_per_launch
            wl[key] = entry
            print(f"{name}: {entry}")
    meta_path.write_text(json.dumps(meta, indent=1) + "\n")
    print("wrote", meta_path)


if __name__ == "__main__":
    main()
