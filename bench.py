#!/usr/bin/env python
"""bench.py -- particles/s of the Count-Sketch update + top-k pass (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg3]

A step = one pass of the whole hot path over the workload's synthetic stream: reset, update (quantise + hash +
red.global scatter), candidate re-scan (estimate every particle's cell against the finished sketch), select,
top-k read-back.  Prints ONE JSON line (rank 0).  `value` = device-resident throughput; `e2e` = the same pass
through the host-streamed C-ABI calls (positions in pinned host memory, H2D copies inside the timed region).
`roofline` is for the dominant kernel (k_update): achieved red.global atomics/s against the measured L2
red rate at the sketch's footprint (cs_probe_l2), with the HBM position-stream term beside it.
`--impl reference` times the CPU oracle, as it stands, on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "particles/sec sketch update+top-k"
UNIT = "particles/s"
REF_SAMPLE = 1 << 21          # particles per step of the --impl reference arm
CPU_BASELINE_SAMPLE = 1 << 23  # particles of the cpu_baseline leg (about 10-30 s of single-core work)

# dram__bytes_read.sum + dram__bytes_write.sum of one k_update launch from the committed `ncu --set full`
# capture (profiles/), keyed by workload; None until a capture exists for that workload.
# thread instructions per particle of the update-phase kernels (smsp__inst_executed.sum x 32 / particles), same capture
NCU_UPDATE_INSTR_PER_PARTICLE = {"cfg3": 425 + 27}
NCU_TRAFFIC_BYTES = {"cfg3": 32.4e9}     # profiles/r1_kernels_cfg3.md: 8 x (scatter + apply) launches per step


def _peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return float(json.loads(p.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def run_oracle_sample(wl, host_xyz, k):
    """One pass of the oracle (update + scan + top-k) over host_xyz; returns seconds."""
    from oracle import cs_oracle as ora
    o = ora.OracleSketch(wl.d, wl.w, wl.G, wl.L, wl.seed)
    t0 = time.perf_counter()
    o.update(host_xyz, wl.sample_p)
    o.scan_begin()
    o.scan(host_xyz, wl.sample_p)
    for s in range(len(wl.G)):
        o.topk(k, s)
    dt = time.perf_counter() - t0
    o.close()
    return dt


def reference_arm(args, wl):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample per step (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_1711_00975_b200 import synth
    n = min(REF_SAMPLE, wl.N)
    host = synth.generate(wl, device="cpu", n=n).numpy()
    k = min(wl.k, n)
    for _ in range(args.warmup):
        run_oracle_sample(wl, host, k)
    t = [run_oracle_sample(wl, host, k) for _ in range(args.steps)]
    total = sum(t)
    value = n * args.steps / total
    sample = f"first {n} particles of the {wl.name} stream per step (same d, w, G, k<= {k}); update + scan + top-k"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": {"workload": wl.name, "N": wl.N, "d": wl.d, "w": wl.w, "G": list(wl.G), "k": wl.k,
                   "sample_p": wl.sample_p, "sampled_particles_per_step": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main_arm(args, wl):
    import torch
    from paper_1711_00975_b200 import binding, sharded, synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA library is the only implementation")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    binding.lib()

    N, p, k = wl.N, wl.sample_p, wl.k
    thr_min = min(wl.thresholds) if wl.thresholds else binding.INT32_MAX
    n_scales = len(wl.G)
    # rank r owns batch r of the stream (same catalogue, per-batch seeds): weak scaling, N particles per GPU
    t_gen = time.perf_counter()
    xyz = synth.generate(wl, device="cuda", batch=rank)
    torch.cuda.synchronize()
    t_gen = time.perf_counter() - t_gen
    checksum = synth.checksum(xyz[: 1 << 20])
    g = binding.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    if args.scan_mode:
        g.set_scan_mode(args.scan_mode)
    if args.update_mode or args.rows_direct != -1:
        g.set_update_mode(args.update_mode, args.rows_direct)

    def step(host=None, ev=None):
        def upd(x, sp):
            if ev:
                ev[0].record()
            (g.update if host is None else g.update_host)(x, sp)
            if ev:
                ev[1].record()
        data = xyz if host is None else host
        res = sharded.sharded_pass(g, data, rank * N, p, k, thr_min, dist, world, update=upd,
                                   scan=g.scan if host is None else g.scan_host,
                                   topk_device="cpu" if host is not None else None)   # e2e: D2H read of the result
        exc = [g.excursion(t, s, cap=0)[2] for s in range(n_scales) for t in wl.thresholds]
        return res, exc

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(nsteps, host=None, upd_events=None):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(nsteps):
            res, _exc = step(host, upd_events[i] if upd_events else None)
        e1.record()
        barrier()
        ms = torch.tensor([e0.elapsed_time(e1)], device="cuda")
        if world > 1:
            dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        return float(ms.item()), res

    # roofline denominators, measured here
    table_bytes = wl.d * wl.w * 4 * n_scales
    ops = 1 << 30
    resident = min(table_bytes, 32 << 20)    # a footprint that stays L2-resident: the PEAK L2 atomic rate
    red_ms = binding.probe_l2(0, resident, ops, reps=3)
    red_fp_ms = binding.probe_l2(0, table_bytes, ops, reps=3)
    gather_ms = binding.probe_l2(2, resident, ops, reps=3)
    stream_ms = binding.probe_stream(xyz, reps=3)
    A_red = ops / (red_ms * 1e-3)            # red.global.add.s32 / s, L2-resident table (BJ's "measured L2 atomic rate")
    A_red_fp = ops / (red_fp_ms * 1e-3)      # the same at the sketch's whole footprint
    A_gather = ops / (gather_ms * 1e-3)
    hbm_peak, hbm_src = _peaks()
    props = torch.cuda.get_device_properties(local)
    sm_count, sm_mhz_max = props.multi_processor_count, 1965.0

    for _ in range(args.warmup):
        step()
    launches0 = g.launch_count()
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    upd_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    ms, res = timed(args.steps, upd_events=upd_ev)
    clk = clocks.stop() if rank == 0 else {}
    launches = g.launch_count() - launches0
    stats = g.scan_stats(0)
    upd_ms = sum(a.elapsed_time(b) for a, b in upd_ev) / args.steps
    ms_per_step = ms / args.steps
    value = world * N / (ms_per_step * 1e-3)

    # end to end: the same pass through the host-streamed calls, positions in pinned host memory
    e2e = None
    if not args.no_e2e:
        host = torch.empty((N, 3), dtype=torch.float32, pin_memory=True)
        host.copy_(xyz)
        torch.cuda.synchronize()
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        step(host)
        ems, eres = timed(e2e_steps, host=host)
        same = all(torch.equal(a[0].cpu(), b[0].cpu()) and torch.equal(a[1].cpu(), b[1].cpu()) for a, b in zip(res, eres))
        e2e = {"value": world * N / (ems / e2e_steps * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 2 * N * 12,
               "d2h_bytes_per_step": sum(int(r[0].numel()) * 12 for r in eres), "steps": e2e_steps,
               "ms_per_step": ems / e2e_steps, "same_result_as_device_path": bool(same)}
        del host

    if rank != 0:
        return
    kept = N * (p if p < 1 else 1.0)
    adds = kept * wl.d * n_scales
    achieved = adds / (upd_ms * 1e-3)
    path_roof = min(hbm_peak * 1e9 / 12.0, A_red / (wl.d * n_scales * (p if p < 1 else 1.0)))
    roofline = {
        "bound": "l2_atomic", "kernel": "update phase (k_bin_scatter + k_bin_apply, or k_update)",
        "achieved": achieved / 1e9, "peak": A_red / 1e9, "unit": "G counter updates/s", "frac": achieved / A_red,
        "traffic": NCU_TRAFFIC_BYTES.get(wl.name),
        "peak_source": f"cs_probe_l2 mode 0 (red.global.add.s32, random addresses) measured in this run on an L2-resident "
                       f"{resident >> 20} MiB table, {ops} ops; at the sketch's {table_bytes >> 20} MiB footprint: "
                       f"{A_red_fp / 1e9:.1f} G/s",
        "algorithmic_units_per_step": adds, "kernel_ms": upd_ms, "kernel_share_of_step": upd_ms / ms_per_step,
        "hbm": {"achieved": N * 12 / (upd_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "frac": N * 12 / (upd_ms * 1e-3) / 1e9 / hbm_peak, "peak_source": hbm_src,
                "stream_only_gbs": N * 12 / (stream_ms * 1e-3) / 1e9},
        "gather_peak_G_per_s": A_gather / 1e9,
        "alu": (None if wl.name not in NCU_UPDATE_INSTR_PER_PARTICLE else {
            "achieved": NCU_UPDATE_INSTR_PER_PARTICLE[wl.name] * N / 32 / (upd_ms * 1e-3) / 1e9,
            "peak": 4 * sm_count * sm_mhz_max * 1e6 / 1e9, "unit": "G warp-instructions/s",
            "frac": NCU_UPDATE_INSTR_PER_PARTICLE[wl.name] * N / 32 / (upd_ms * 1e-3) / (4 * sm_count * sm_mhz_max * 1e6),
            "peak_source": "4 warp schedulers per SM x SM count x max SM clock (B200_PROFILING.md: 148 SMs, 1965 MHz); "
                           "instruction counts from profiles/r1_kernels_cfg3.md"}),
        "path": {"roof_particles_per_s": path_roof, "frac": (value / world) / path_roof,
                 "formula": "min(HBM/12B, A_L2/(d*scales*p)) per GPU, whole update+scan+select step against it "
                            "(BASELINE.json north_star)"},
    }
    cpu = None
    if not args.no_cpu_baseline:
        n_s = min(CPU_BASELINE_SAMPLE, N)
        hs = xyz[:n_s].cpu().numpy()
        dt = run_oracle_sample(wl, hs, min(k, n_s))
        cpu = {"value": n_s / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
               "sample": f"first {n_s} particles of the {wl.name} stream, same d/w/G, k={min(k, n_s)}: update + scan + top-k, "
                         f"single thread; host has {os.cpu_count()} cores"}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32", "data": "synthetic",
        "config": {"workload": wl.name, "N_per_gpu": N, "d": wl.d, "w": wl.w, "G": list(wl.G), "k": k, "sample_p": p,
                   "thresholds": list(wl.thresholds), "l2_between_iterations": "inputs (12 B x N) larger than L2",
                   "positions_checksum_first_2^20": checksum, "generate_s": t_gen,
                   "parallelism": "stream shards + int32 table all-reduce + top-k all-gather" if world > 1 else "1 GPU"},
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clk,
        "scan": {"candidates": stats["candidates"], "tau": stats["tau"], "compactions": stats["compactions"],
                 "scan_launches": stats["scan_launches"], "topk_returned": [int(r[0].numel()) for r in res]},
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def streamed_arm(args, wl):
    """Workloads that do not fit the device (cfg 4: 10^10 particles = 120 GB): the stream lives in pinned host memory
    (generated batch by batch on the device with per-batch keys, copied out once, untimed) and every step goes
    through cs_update_host / cs_scan_host, i.e. `value` IS the end-to-end number: H2D copies inside the timed region."""
    import torch
    from paper_1711_00975_b200 import binding, sharded, synth

    if int(os.environ.get("WORLD_SIZE", "1")) != 1:
        raise SystemExit("the host-streamed workload runs on one GPU")
    torch.cuda.set_device(0)
    binding.lib()
    N, B = (args.n or wl.N), wl.batch
    k, p = wl.k, wl.sample_p
    packed = args.packed               # 8-byte records (cs_pack_records) instead of 12-byte float32 positions
    bpp = 8 if packed else 12
    g = binding.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    t0 = time.perf_counter()
    host = (torch.empty(N, dtype=torch.int64, pin_memory=True) if packed
            else torch.empty((N, 3), dtype=torch.float32, pin_memory=True))
    t_pin = time.perf_counter() - t0
    cat = synth.Catalogue(wl, "cuda")
    t0 = time.perf_counter()
    checksum = None
    for b, lo in enumerate(range(0, N, B)):
        m = min(B, N - lo)
        xb = synth.generate(wl, device="cuda", batch=b, n=m, catalogue=cat)
        if checksum is None:
            checksum = synth.checksum(xb[: 1 << 20])
        host[lo:lo + m].copy_(g.pack_records(xb) if packed else xb)
        del xb
    torch.cuda.synchronize()
    t_gen = time.perf_counter() - t0
    # pinned H2D bandwidth: the stream term of this workload's roofline
    probe_n = min(N, 1 << 28)
    dev = torch.empty_like(host[:probe_n], device="cuda")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dev.copy_(host[:probe_n], non_blocking=True)
    e0.record()
    for _ in range(3):
        dev.copy_(host[:probe_n], non_blocking=True)
    e1.record()
    torch.cuda.synchronize()
    h2d_gbs = 3 * probe_n * bpp / (e0.elapsed_time(e1) * 1e-3) / 1e9
    del dev

    def step(ev=None):
        def upd(x, sp):
            if ev:
                ev[0].record()
            (g.update_records_host if packed else g.update_host)(x, sp)
            if ev:
                ev[1].record()
        return sharded.sharded_pass(g, host, 0, p, k, binding.INT32_MAX, update=upd,
                                    scan=g.scan_records_host if packed else g.scan_host, topk_device="cpu")

    for _ in range(args.warmup):
        step()
    launches0 = g.launch_count()
    clocks = ClockSampler(0)
    clocks.start()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    e0.record()
    for i in range(args.steps):
        res = step(ev[i])
    e1.record()
    torch.cuda.synchronize()
    clk = clocks.stop()
    ms_per_step = e0.elapsed_time(e1) / args.steps
    upd_ms = sum(a.elapsed_time(b) for a, b in ev) / args.steps
    value = N / (ms_per_step * 1e-3)
    stats = g.scan_stats(0)
    roof = h2d_gbs * 1e9 / bpp / 2.0        # the stream crosses PCIe twice per step (update, re-scan)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32",
        "data": "synthetic",
        "config": {"workload": wl.name, "N": N, "d": wl.d, "w": wl.w, "G": list(wl.G), "k": k, "sample_p": p,
                   "batches": (N + B - 1) // B, "host_streamed": True,
                   "input": "packed 64-bit records (integer cell rule, cs.h)" if packed else "float32 xyz",
                   "l2_between_iterations": "inputs (12 B x N) larger than L2", "positions_checksum_first_2^20": checksum,
                   "pin_s": t_pin, "generate_s": t_gen, "parallelism": "1 GPU"},
        "roofline": {"bound": "pcie", "kernel": "cs_update_host (H2D ring + update kernels)",
                     "achieved": N * bpp / (upd_ms * 1e-3) / 1e9, "peak": h2d_gbs, "unit": "GB/s",
                     "frac": N * bpp / (upd_ms * 1e-3) / 1e9 / h2d_gbs, "traffic": None,
                     "peak_source": "pinned host -> device copy of 2^28-particle blocks measured in this run",
                     "kernel_ms": upd_ms, "kernel_share_of_step": upd_ms / ms_per_step,
                     "path": {"roof_particles_per_s": roof, "frac": value / roof,
                              "formula": f"PCIe bandwidth / {bpp} B / 2 passes (BASELINE.json north_star: PCIe for host-streamed runs)"}},
        "cpu_baseline": None,
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 2 * N * bpp,
                "d2h_bytes_per_step": sum(int(r[0].numel()) * 12 for r in res), "steps": args.steps, "ms_per_step": ms_per_step},
        "gpu_launches": g.launch_count() - launches0, "clocks": clk,
        "scan": {"candidates": stats["candidates"], "tau": stats["tau"], "compactions": stats["compactions"],
                 "scan_launches": stats["scan_launches"], "topk_returned": [int(r[0].numel()) for r in res]},
        "context": "paper: top 3e5 cells of 1e10 particles on a ~1e11-cell grid in < 5 min on one GTX 1080 / Tesla C2050 "
                   "(PAPER.md:31, :314)",
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--n", type=int, default=0, help="override the particle count (debugging; not a bench value)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--packed", action="store_true", help="host-streamed workloads: 8-byte packed records instead of float32 xyz")
    ap.add_argument("--scan-mode", type=int, default=0, help="cs_set_scan_mode: 0 auto, 1 plain, 2 bitmap, 3 bitmap stages")
    ap.add_argument("--update-mode", type=int, default=0, help="cs_set_update_mode: 0 auto, 1 direct, 2 binned")
    ap.add_argument("--rows-direct", type=int, default=-1, help="rows of each binned pass that use red.global")
    args = ap.parse_args()
    from paper_1711_00975_b200 import synth
    wl = synth.CONFIGS[args.workload]
    if args.n and not wl.batch:
        wl = wl.scaled(args.n)
    if args.impl == "reference":
        reference_arm(args, wl)
    elif wl.batch:
        streamed_arm(args, wl)
    else:
        main_arm(args, wl)


if __name__ == "__main__":
    main()
