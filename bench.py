#!/usr/bin/env python
"""bench.py -- particles/s of the Count-Sketch update + top-k pass (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg3]
    python bench.py --sweep            # roofline denominators: L2 red / atom / gather vs footprint, PCIe

A step = one pass of the whole hot path over the workload's synthetic stream: reset, update (quantise + hash +
scatter), candidate re-scan (estimate every particle's cell against the finished sketch), select, top-k read-back.
Prints ONE JSON line (rank 0).
  value      device-resident throughput (positions already in HBM), whole job, max over ranks.
  e2e        the same pass through the host-streamed C-ABI calls: positions in pinned host memory, H2D copies and the
             D2H read of the result inside the timed region.
  roofline   for the dominant kernel (the update's scatter kernel): achieved warp-instruction rate against the issue
             peak of the chip ("bound": "alu" -- the kernel is hashing arithmetic), its duration
             measured live with CUDA events the library records on its own stream (cs_set_timing); instruction count
             and DRAM traffic per launch come from the committed ncu capture profiles/r2_kernel_metrics.json and are
             null when the kernel sources have changed since that capture.  roofline.path = the whole step against
             BASELINE.json's contract roofline min(HBM / 12 B, A_L2 / (d * scales * p)).
  cpu_baseline  the oracle as it stands on one host core, bounded sample, best of 3, update and scan+select apart.
`--impl reference` times the CPU oracle, as it stands, on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import hashlib
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
REF_SAMPLE = 1 << 21           # particles per step of the --impl reference arm
CPU_BASELINE_SAMPLE = 1 << 22  # particles of the cpu_baseline leg: 3 repetitions of ~6 s of single-core work
SM_MAX_MHZ = 1965.0            # B200_PROFILING.md: clocks.max.sm
CAPTURE = ROOT / "profiles" / "r2_kernel_metrics.json"
KERNEL_SOURCES = ["cs_update_binned.cu", "cs_hash.h", "cs_device.cuh", "cs_internal.h", "cs_scan_staged.cu",
                  "cs_scan_common.cuh"]


def _peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return float(json.loads(p.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def kernel_sources_sha() -> str:
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        h.update((ROOT / "paper_1711_00975_b200" / "csrc" / f).read_bytes())
    return h.hexdigest()[:16]


def load_capture(workload: str):
    """ncu-derived per-launch figures of the hot kernels for this workload, or None when there is no capture of the
    kernel sources as they stand (profiles/r2_kernel_metrics.json names the sources' hash it was taken on)."""
    try:
        c = json.loads(CAPTURE.read_text())
    except Exception:
        return None
    if c.get("kernel_sources_sha") != kernel_sources_sha():
        return None
    return c.get("workloads", {}).get(workload)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region.  power.draw is not queried: with it, about one
    run in eight of cfg 5 (5 steps of 20 ms) had a step stretched by ~25 ms -- the query holds a driver lock that kernel
    launches wait for (8 runs without any sampling: 19.6-20.3 ms; 24 runs with this query: 19.6-21.6 ms)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int, interval_ms: int = 100, source: str = "nvidia-smi"):
        self.index, self.rows, self.proc, self.interval_ms, self.source = index, [], None, interval_ms, source
        self.live = False

    def _nvml_loop(self, nv, h, mx):
        bits = [nv.nvmlClocksThrottleReasonHwSlowdown, nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                nv.nvmlClocksThrottleReasonSwThermalSlowdown, nv.nvmlClocksThrottleReasonSwPowerCap]
        while self.live:
            try:
                sm = nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                self.rows.append((time.monotonic(), [str(sm), str(mx)] + ["Active" if r & b else "Not Active" for b in bits]))
            except Exception:
                pass
            time.sleep(self.interval_ms / 1000.0)

    def start(self):
        if self.interval_ms <= 0:
            return
        if self.source == "nvml":                       # the library nvidia-smi reads, in this process (no start-up, one
            try:                                        # clock and one reasons query per sample)
                import pynvml as nv
                nv.nvmlInit()
                h = nv.nvmlDeviceGetHandleByIndex(self.index)
                mx = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
                self.live = True
                self.proc = threading.Thread(target=self._nvml_loop, args=(nv, h, mx), daemon=True)
                self.proc.start()
                return
            except Exception:
                self.live, self.proc, self.source = False, None, "nvidia-smi"
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", str(self.interval_ms)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
            # nvidia-smi holds driver locks while it starts (about a second): kernel launches issued meanwhile stall, which
            # showed as an occasional 25 instead of 20 ms per step on cfg 5.  Wait for its first sample before any step.
            t_end = time.monotonic() + 5.0
            while not self.rows and time.monotonic() < t_end and self.proc.poll() is None:
                time.sleep(0.01)
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.monotonic(), [c.strip() for c in line.split(",")]))

    def mark(self):
        """Start of the timed region: only samples taken after this count.  (The sampler itself is started before the
        warm-up steps: the start-up of nvidia-smi takes driver locks for about a second and would otherwise stretch the
        first timed steps of a short run -- measured: cfg 5, 5 steps, 25.6 instead of 20.3 ms per step.)"""
        self.t0 = time.monotonic()

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05 + self.interval_ms / 1000.0)
        if self.live:
            self.live = False
        else:
            self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, r in self.rows:
            if t < getattr(self, "t0", 0.0):
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for nm, v in zip(names, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "source": self.source}


def run_oracle_sample(wl, host_xyz, k):
    """One pass of the oracle over host_xyz; returns (update seconds, scan + select seconds)."""
    from oracle import cs_oracle as ora
    o = ora.OracleSketch(wl.d, wl.w, wl.G, wl.L, wl.seed)
    t0 = time.perf_counter()
    o.update(host_xyz, wl.sample_p)
    t1 = time.perf_counter()
    o.scan_begin()
    o.scan(host_xyz, wl.sample_p)
    for s in range(len(wl.G)):
        o.topk(k, s)
        for thr in wl.thresholds:
            o.excursion(thr, s)
    t2 = time.perf_counter()
    o.close()
    return t1 - t0, t2 - t1


def cpu_baseline(wl, host_xyz, k, reps=3):
    runs = [run_oracle_sample(wl, host_xyz, k) for _ in range(reps)]
    upd, sel = min(r[0] for r in runs), min(r[1] for r in runs)
    n = len(host_xyz)
    return {"value": n / (upd + sel), "unit": UNIT, "cores": 1, "kind": "oracle", "best_of": reps,
            "update_s": upd, "scan_select_s": sel, "update_particles_per_s": n / upd,
            "scan_select_particles_per_s": n / sel,
            "sample": f"first {n} particles of the {wl.name} stream, same d/w/G/p, k={k}: update, then scan + top-k"
                      f"{' + excursion sets' if wl.thresholds else ''}; single thread, best of {reps}; host has "
                      f"{os.cpu_count()} cores"}


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
    t = [sum(run_oracle_sample(wl, host, k)) for _ in range(args.steps)]
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


def _roofline(wl, world, N, value, ms_per_step, phases, hbm_peak, hbm_src, A_red, A_red_fp, A_gather, stream_ms, resident,
              table_bytes, sm_count, n_rows_direct_note):
    """The roofline object of the contract, for the dominant kernel (update scatter) + the information bounds."""
    p = wl.sample_p if wl.sample_p < 1 else 1.0
    n_scales = len(wl.G)
    kept = N * p
    cap = load_capture(wl.name)
    sc_ms, sc_n = phases["update_scatter"]
    ap_ms, _ = phases["update_apply"]
    kernel_ms = sc_ms / sc_n if sc_n else None
    issue_peak = 4 * sm_count * SM_MAX_MHZ * 1e6 / 1e9           # G warp-instructions/s
    achieved = traffic = instr = None
    if cap and sc_ms > 0:
        instr = cap["k_bin_scatter"]["thread_instructions_per_particle"]
        achieved = instr * kept * cap["k_bin_scatter"]["passes_per_particle"] / 32 / (sc_ms * 1e-3) / 1e9
        traffic = cap["k_bin_scatter"]["dram_bytes_per_launch"]
    upd_ms = sc_ms + ap_ms + phases["compact_kept"][0] / 2.0
    path_roof = min(hbm_peak * 1e9 / 12.0, A_red / (wl.d * n_scales * p))
    return {
        "bound": "alu", "kernel": "k_bin_scatter (update: quantise + 2d hashes + record scatter; or k_update in direct mode)",
        "achieved": achieved, "peak": issue_peak, "unit": "G warp-instructions/s",
        "frac": (achieved / issue_peak) if achieved else None, "traffic": traffic,
        "peak_source": f"4 warp schedulers x {sm_count} SMs x {SM_MAX_MHZ:.0f} MHz (B200_PROFILING.md unit counts and clocks; "
                       "DESIGN.md section 6.2)",
        "achieved_source": ("thread instructions per particle and DRAM bytes per launch from " + CAPTURE.name +
                            " (ncu capture of these kernel sources)") if cap else
                           "null: no ncu capture of the kernel sources as they stand (profiles/r2_kernel_metrics.json)",
        "thread_instructions_per_particle": instr,
        "kernel_ms": kernel_ms, "kernel_launches_per_step": sc_n, "kernel_ms_per_step": sc_ms,
        "kernel_share_of_step": sc_ms / ms_per_step if ms_per_step else None,
        "phases_ms_per_step": {k: v[0] for k, v in phases.items() if v[1]},
        "phase_launch_groups_per_step": {k: v[1] for k, v in phases.items() if v[1]},
        "hbm": {"achieved": N * 12 / (upd_ms * 1e-3) / 1e9 if upd_ms else None, "peak": hbm_peak, "unit": "GB/s",
                "frac": N * 12 / (upd_ms * 1e-3) / 1e9 / hbm_peak if upd_ms else None, "peak_source": hbm_src,
                "what": "12 B/particle of the update phase against the copy bandwidth",
                "stream_only_gbs": N * 12 / (stream_ms * 1e-3) / 1e9},
        "l2_atomic": {"peak_resident_G_per_s": A_red / 1e9, "peak_at_footprint_G_per_s": A_red_fp / 1e9,
                      "resident_table_MiB": resident >> 20, "footprint_MiB": table_bytes >> 20,
                      "gather_peak_G_per_s": A_gather / 1e9,
                      "counter_updates_per_s_G": kept * wl.d * n_scales / (upd_ms * 1e-3) / 1e9 if upd_ms else None,
                      "note": "counter updates/s of the update phase can exceed the red.global peak: " + n_rows_direct_note},
        "path": {"roof_particles_per_s": path_roof, "frac": (value / world) / path_roof, "hard_bound": False,
                 "formula": "min(HBM/12B, A_L2/(d*scales*p)) per GPU with A_L2 = the L2-resident red.global.add peak "
                            "measured in this run; the whole update+scan+select step against it (BASELINE.json north_star)",
                 "note": "the contract's denominator, not a hard bound of this design: the update sends 4 of 7 rows through "
                         "shared-memory atomics instead of L2 atomics, so the step can come close to (or pass) A_L2/d"},
    }


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

    strong = args.scaling == "strong" and world > 1
    p, k = wl.sample_p, wl.k
    thr_min = min(wl.thresholds) if wl.thresholds else binding.INT32_MAX
    n_scales = len(wl.G)
    t_gen = time.perf_counter()
    if strong:      # one stream of wl.N particles cut into contiguous shards (total work fixed)
        lo, hi = sharded.shard_bounds(wl.N, rank, world)
        cat = synth.Catalogue(wl, "cuda")
        xyz = torch.empty((hi - lo, 3), dtype=torch.float32, device="cuda")
        for i0 in range(lo, hi, 1 << 22):                    # chunked: the generator holds ~20 temporaries per particle
            m = min(1 << 22, hi - i0)
            cat.positions(i0, m, out=xyz[i0 - lo:i0 - lo + m])
        index0 = lo
    else:           # rank r owns batch r of the stream (same catalogue, per-batch keys): N particles per GPU
        xyz = synth.generate(wl, device="cuda", batch=rank)
        index0 = rank * wl.N
    N = xyz.shape[0]
    torch.cuda.synchronize()
    t_gen = time.perf_counter() - t_gen
    checksum = synth.checksum(xyz[: 1 << 20])
    g = binding.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    if args.scan_mode:
        g.set_scan_mode(args.scan_mode)
    if args.update_mode or args.rows_direct != -1:
        g.set_update_mode(args.update_mode, args.rows_direct)
    replay_bytes = 0
    if p < 0.5 and not args.no_replay_cache:     # sampled stream: the re-scan reuses the kept particles of the update
        replay_bytes = int(N * p * 12 * 2.5) + (64 << 20)
        g.set_replay_cache(replay_bytes)

    def step(host=None, ev=None):
        def upd(x, sp):
            if ev:
                ev[0].record()
            (g.update if host is None else g.update_host)(x, sp)
            if ev:
                ev[1].record()
        data = xyz if host is None else host
        res = sharded.sharded_pass(g, data, index0, p, k, thr_min, dist, world, update=upd,
                                   scan=g.scan if host is None else g.scan_host,
                                   topk_device="cpu" if host is not None else None)   # e2e: D2H read of the result
        exc = [g.excursion(t, s, cap=0)[2] for s in range(n_scales) for t in wl.thresholds]
        return res, exc

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(nsteps, host=None, upd_events=None):
        import gc
        gc.collect()          # keep interpreter collections out of the timed region (cfg 5: 100 ms in all)
        gc.disable()
        try:
            return _timed(nsteps, host, upd_events)
        finally:
            gc.enable()

    def _timed(nsteps, host=None, upd_events=None):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(nsteps):
            res, exc = step(host, upd_events[i] if upd_events else None)
        e1.record()
        barrier()
        ms = torch.tensor([e0.elapsed_time(e1)], device="cuda")
        if world > 1:
            dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        return float(ms.item()), res, exc

    # roofline denominators, measured here
    table_bytes = wl.d * wl.w * 4 * n_scales
    ops = 1 << 30
    resident = min(table_bytes, 32 << 20)    # a footprint that stays L2-resident: the PEAK L2 atomic rate
    red_ms = binding.probe_l2(0, resident, ops, reps=3)
    red_fp_ms = binding.probe_l2(0, table_bytes, ops, reps=3)
    gather_ms = binding.probe_l2(2, resident, ops, reps=3)
    stream_ms = binding.probe_stream(xyz, reps=3)
    A_red, A_red_fp, A_gather = ops / (red_ms * 1e-3), ops / (red_fp_ms * 1e-3), ops / (gather_ms * 1e-3)
    hbm_peak, hbm_src = _peaks()
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count

    clocks = ClockSampler(local, args.clock_interval_ms, args.clock_source)
    if rank == 0:
        clocks.start()
    for _ in range(args.warmup):
        step()
    g.update_stats()
    launches0 = g.launch_count()
    clocks.mark()
    upd_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    ms, res, exc = timed(args.steps, upd_events=upd_ev)
    clk = clocks.stop() if rank == 0 else {}
    launches = g.launch_count() - launches0
    routes = g.update_stats()
    stats = [g.scan_stats(s) for s in range(n_scales)]
    upd_ms = sum(a.elapsed_time(b) for a, b in upd_ev) / args.steps
    ms_per_step = ms / args.steps
    total_particles = wl.N if strong else world * N
    value = total_particles / (ms_per_step * 1e-3)

    # per-kernel-class device times: separate steps with the library's event recording on (not part of `value`)
    psteps = max(1, min(3, args.steps))
    g.set_timing(True)
    for _ in range(psteps):
        step()
    tm = g.get_timing()
    g.set_timing(False)
    phases = {kk: (v[0] / psteps, v[1] / psteps) for kk, v in tm.items()}

    # end to end: the same pass through the host-streamed calls, positions in pinned host memory
    e2e = None
    if not args.no_e2e:
        host = torch.empty((N, 3), dtype=torch.float32, pin_memory=True)
        host.copy_(xyz)
        torch.cuda.synchronize()
        e2e_steps = max(1, min(args.steps, args.e2e_steps))

        def same(a, b):
            return all(torch.equal(x[0].cpu(), y[0].cpu()) and torch.equal(x[1].cpu(), y[1].cpu()) for x, y in zip(a, b))
        step(host)
        ems2, eres2, _ = timed(e2e_steps, host=host)          # staging ring: update and re-scan both cross PCIe
        two = {"value": total_particles / (ems2 / e2e_steps * 1e-3), "ms_per_step": ems2 / e2e_steps,
               "h2d_bytes_per_step": 2 * N * 12, "same_result_as_device_path": bool(same(res, eres2))}
        free, _tot = torch.cuda.mem_get_info()
        one = None
        if free > N * 12 + (8 << 30) and not args.no_replay_cache:
            g.set_replay_cache(N * 12 + replay_bytes + (64 << 20))   # the re-scan reads the device copy of the update
            step(host)
            ems1, eres1, _ = timed(e2e_steps, host=host)
            one = {"value": total_particles / (ems1 / e2e_steps * 1e-3), "ms_per_step": ems1 / e2e_steps,
                   "h2d_bytes_per_step": N * 12, "same_result_as_device_path": bool(same(res, eres1))}
            g.set_replay_cache(replay_bytes)
        best = one or two
        e2e = {"value": best["value"], "unit": UNIT, "h2d_bytes_per_step": best["h2d_bytes_per_step"],
               "d2h_bytes_per_step": sum(int(r[0].numel()) * 12 for r in eres2), "steps": e2e_steps,
               "ms_per_step": best["ms_per_step"], "same_result_as_device_path": best["same_result_as_device_path"],
               "how": ("cs_set_replay_cache: cs_update_host copies the stream to the device once, cs_scan_host re-scans that copy"
                       if one else "staging ring: update and re-scan both stream the positions from pinned host memory"),
               "two_crossings": two}
        del host

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    total_routes = max(1, sum(routes.values()))
    note = ("rows that take the binned route are applied with shared-memory atomics, not L2 atomics "
            f"(routes of the binned rows this run: {routes})")
    roofline = _roofline(wl, world, N, value, ms_per_step, phases, hbm_peak, hbm_src, A_red, A_red_fp, A_gather, stream_ms,
                         resident, table_bytes, sm_count, note)
    roofline["update_phase_ms"] = upd_ms
    cpu = None
    if not args.no_cpu_baseline:
        n_s = min(CPU_BASELINE_SAMPLE, N)
        cpu = cpu_baseline(wl, xyz[:n_s].cpu().numpy(), min(k, n_s))
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if strong else "weak", "vs_baseline": None,
        "dtype": "int32", "data": "synthetic",
        "config": {"workload": wl.name, "N_per_gpu": N, "N_total": total_particles, "d": wl.d, "w": wl.w, "G": list(wl.G),
                   "k": k, "sample_p": p, "thresholds": list(wl.thresholds), "sigma_mult": wl.sigma_mult,
                   "l2_between_iterations": "inputs (12 B x N) larger than L2" if N * 12 > (126 << 20) else
                                            "none: inputs smaller than L2 (small config, not the headline)",
                   "positions_checksum_first_2^20": checksum, "generate_s": t_gen, "replay_cache_bytes": replay_bytes,
                   "parallelism": "stream shards + int32 table all-reduce + top-k all-gather" if world > 1 else "1 GPU"},
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clk,
        "update_routes": {**routes, "overflow_share": (routes["staging_overflow"] + routes["region_overflow"]) / total_routes},
        "scan": {"per_scale": stats, "topk_returned": [int(r[0].numel()) for r in res], "excursion_sizes": exc},
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def streamed_arm(args, wl):
    """Workloads that do not fit the device (cfg 4: 10^10 particles = 120 GB): the stream lives in pinned host memory
    (generated batch by batch on the device with per-batch keys, copied out once, untimed) and every step goes
    through cs_update_host / cs_scan_host, i.e. `value` IS the end-to-end number: H2D copies inside the timed region.
    --query hierarchical: one crossing -- the update feeds a coarse and the fine mesh at once, the query is the paper's
    positions-free two-layer search (Alg. 3) over ALL cells of the coarse mesh and the children
    of its heavy cells: a different candidate set (full dictionary, not the occupied cells), stated in the line."""
    import torch
    from paper_1711_00975_b200 import binding, sharded, synth

    if int(os.environ.get("WORLD_SIZE", "1")) != 1:
        raise SystemExit("the host-streamed workload runs on one GPU")
    torch.cuda.set_device(0)
    binding.lib()
    N, B = (args.n or wl.N), wl.batch
    k, p = wl.k, wl.sample_p
    packed = args.packed               # 8-byte records (cs_pack_records) instead of 12-byte float32 positions
    hier = args.query == "hierarchical"
    bpp = 8 if packed else 12
    Gs = list(wl.G)
    if hier:                           # coarse layer of super-cells of r^3 cells, r the divisor of G nearest 10 (paper: ~10^3)
        r = min((q for q in range(2, 65) if wl.G[0] % q == 0), key=lambda q: abs(q - 10))
        Gs = [wl.G[0] // r, wl.G[0]]
    g = binding.CountSketch(wl.d, wl.w, Gs, wl.L, wl.seed)
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
        if ev:
            ev[0].record()
        if not hier:
            def upd(x, sp):
                (g.update_records_host if packed else g.update_host)(x, sp)
                if ev:
                    ev[1].record()
            return sharded.sharded_pass(g, host, 0, p, k, binding.INT32_MAX, update=upd,
                                        scan=g.scan_records_host if packed else g.scan_host, topk_device="cpu")
        g.reset()
        (g.update_records_host if packed else g.update_host)(host, p)
        if ev:
            ev[1].record()
        g.scan_begin(4 * k)                                  # Alg. 3: the c*k heaviest super-cells, c = 4
        g.scan_all(0)
        parents, _ = g.topk(4 * k, 0)
        g.scan_children(parents, 0, 1)
        return [g.topk(k, 1, device="cpu")]

    clocks = ClockSampler(0, args.clock_interval_ms, args.clock_source)
    clocks.start()
    for _ in range(args.warmup):
        step()
    launches0 = g.launch_count()
    torch.cuda.synchronize()
    clocks.mark()
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
    stats = g.scan_stats(1 if hier else 0)
    crossings = 1 if hier else 2
    roof = h2d_gbs * 1e9 / bpp / crossings
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32",
        "data": "synthetic",
        "config": {"workload": wl.name, "N": N, "d": wl.d, "w": wl.w, "G": Gs, "k": k, "sample_p": p,
                   "batches": (N + B - 1) // B, "host_streamed": True,
                   "input": "packed 64-bit records (integer cell rule, cs.h)" if packed else "float32 xyz",
                   "query": ("hierarchical, positions-free (Alg. 3): full search of the coarse mesh, children of its "
                             f"{4 * k} heaviest cells; candidate set = full dictionary, NOT the occupied cells of the re-scan")
                            if hier else "candidate re-scan of the replayed stream (BASELINE.json north_star)",
                   "l2_between_iterations": "inputs (12 B x N) larger than L2", "positions_checksum_first_2^20": checksum,
                   "pin_s": t_pin, "generate_s": t_gen, "parallelism": "1 GPU"},
        "roofline": {"bound": "pcie", "kernel": "cs_update_host (H2D ring + update kernels)",
                     "achieved": N * bpp / (upd_ms * 1e-3) / 1e9, "peak": h2d_gbs, "unit": "GB/s",
                     "frac": N * bpp / (upd_ms * 1e-3) / 1e9 / h2d_gbs, "traffic": None,
                     "peak_source": "pinned host -> device copy of 2^28-particle blocks measured in this run",
                     "kernel_ms": upd_ms, "kernel_share_of_step": upd_ms / ms_per_step,
                     "path": {"roof_particles_per_s": roof, "frac": value / roof,
                              "formula": f"PCIe bandwidth / {bpp} B / {crossings} crossing(s) (BASELINE.json north_star: "
                                         "PCIe for host-streamed runs)"}},
        "cpu_baseline": None,
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": crossings * N * bpp,
                "d2h_bytes_per_step": sum(int(r[0].numel()) * 12 for r in res), "steps": args.steps, "ms_per_step": ms_per_step},
        "gpu_launches": g.launch_count() - launches0, "clocks": clk,
        "scan": {"candidates": stats["candidates"], "tau": stats["tau"], "compactions": stats["compactions"],
                 "scan_launches": stats["scan_launches"], "topk_returned": [int(r[0].numel()) for r in res]},
        "context": "paper: top 3e5 cells of 1e10 particles on a ~1e11-cell grid in < 5 min on one GTX 1080 / Tesla C2050 "
                   "(PAPER.md:31, :314)",
    }
    print(json.dumps(line), flush=True)


def sweep_arm(args):
    """SURVEY 8.d.3 microbenchmarks that define the roofline denominators: red.global.add / returning atom / 4-byte
    gathers at random addresses over tables of the BASELINE.json sketch footprints, and pinned H2D copies alone and
    with a concurrent D2H."""
    import torch
    from paper_1711_00975_b200 import binding
    torch.cuda.set_device(0)
    binding.lib()
    ops = 1 << 29
    rows = []
    for mib in (1.25, 16, 20, 80, 112, 320, 448):
        nbytes = int(mib * (1 << 20))
        r = {"table_MiB": mib}
        for mode, name in ((0, "red_G_per_s"), (1, "atom_G_per_s"), (2, "gather_G_per_s")):
            r[name] = ops / (binding.probe_l2(mode, nbytes, ops, reps=3) * 1e-3) / 1e9
        rows.append(r)
    n = (1 << 28) * 12                                        # 3.2 GB blocks
    h = torch.empty(n, dtype=torch.uint8, pin_memory=True)
    h2 = torch.empty(n, dtype=torch.uint8, pin_memory=True)
    d = torch.empty(n, dtype=torch.uint8, device="cuda")
    d2 = torch.empty(n, dtype=torch.uint8, device="cuda")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()

    def copy_rate(with_d2h):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        with torch.cuda.stream(s1):
            e0.record()
            for _ in range(3):
                d.copy_(h, non_blocking=True)
            e1.record()
        if with_d2h:
            with torch.cuda.stream(s2):
                for _ in range(3):
                    h2.copy_(d2, non_blocking=True)
        torch.cuda.synchronize()
        return 3 * n / (e0.elapsed_time(e1) * 1e-3) / 1e9
    copy_rate(False)
    pcie = {"h2d_alone_GB_per_s": copy_rate(False), "h2d_with_concurrent_d2h_GB_per_s": copy_rate(True), "block_GB": n / 1e9}
    hbm_peak, hbm_src = _peaks()
    print(json.dumps({"sweep": "SURVEY 8.d.3 roofline denominators", "ops_per_point": ops, "l2": rows, "pcie": pcie,
                      "hbm_copy_GB_per_s": hbm_peak, "hbm_source": hbm_src}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = the workload's N per GPU (default); strong = one stream of N cut into shards")
    ap.add_argument("--n", type=int, default=0, help="override the particle count (debugging; not a bench value)")
    ap.add_argument("--sigma-mult", type=float, default=1.0,
                    help="< 1: the concentrated stress variant of the generator (SURVEY 8.d.2 iii); never a BASELINE config")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-replay-cache", action="store_true")
    ap.add_argument("--packed", action="store_true", help="host-streamed workloads: 8-byte packed records instead of float32 xyz")
    ap.add_argument("--query", default="rescan", choices=["rescan", "hierarchical"],
                    help="host-streamed workloads: hierarchical = positions-free two-layer query, one PCIe crossing")
    ap.add_argument("--scan-mode", type=int, default=0, help="cs_set_scan_mode: 0 auto, 1 plain, 2 bitmap, 3 bitmap stages")
    ap.add_argument("--update-mode", type=int, default=0, help="cs_set_update_mode: 0 auto, 1 direct, 2 binned")
    ap.add_argument("--rows-direct", type=int, default=-1, help="rows of each binned pass that use red.global")
    ap.add_argument("--clock-interval-ms", type=int, default=100,
                    help="nvidia-smi sampling period during the timed region (100: the timed region of cfg 5 lasts 100 ms); "
                         "0 = no sampling (debugging)")
    ap.add_argument("--clock-source", default="nvidia-smi", choices=["nvidia-smi", "nvml"])
    ap.add_argument("--sweep", action="store_true", help="print the roofline-denominator sweep instead of a bench line")
    args = ap.parse_args()
    if args.sweep:
        return sweep_arm(args)
    from paper_1711_00975_b200 import synth
    wl = synth.CONFIGS[args.workload]
    if args.n and not wl.batch:
        wl = wl.scaled(args.n)
    if args.sigma_mult != 1.0:
        wl = wl.scaled(wl.N, sigma_mult=args.sigma_mult)
    if args.impl == "reference":
        reference_arm(args, wl)
    elif wl.batch:
        streamed_arm(args, wl)
    else:
        main_arm(args, wl)


if __name__ == "__main__":
    main()
