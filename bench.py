#!/usr/bin/env python
"""bench.py -- device-resident throughput of the F-engine path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]

A "step" is one fengine_process call over one synthetic batch of BASELINE.json configs[1]
(4 antennas x 2 pols, n=4096, T=16, 2^24 samples per pol): all hot-path rows of SURVEY.md section 8(a).
`value` = dual-pol sample instants turned into output per second (Gsample/s dual-pol = A*S*N / t),
inputs resident in HBM.  `e2e` is the same metric through fengine_process_host with pinned HOST buffers
(H2D + path + D2H inside the timed region).  One JSON line is printed by rank 0.

--impl reference times the float64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "Gsample/s dual-pol, device-resident, n=4096 T=16; % of HBM roofline"
UNIT = "Gsample/s"
ALG_BYTES_PER_DUALPOL_SAMPLE = 4.5     # 1.25 B in + 1 B out per real sample, x2 pols


def csrc_hash() -> str:
    """sha256 over the kernel sources (sorted by name): ties profiles/roofline_traffic.csv to the code it measured."""
    import hashlib
    h = hashlib.sha256()
    for f in sorted((ROOT / "paper_2303_09886_b200" / "csrc").glob("*.cu*")):
        h.update(f.name.encode())
        h.update(f.read_bytes())
    return h.hexdigest()


def workload_stamp(args, w=None) -> str:
    """What was measured, as one string: the second stamp of profiles/roofline_traffic.csv (the ncu capture there is of
    ONE workload and option set; a run of anything else must not report its DRAM bytes)."""
    opts = sorted(args.opt)
    if args.chunk_spectra is not None:
        opts.append(f"chunk_spectra={args.chunk_spectra}")
    if args.fir_rows is not None:
        opts.append(f"fir_rows={args.fir_rows}")
    if getattr(args, "pol_offset", 0):
        opts.append(f"pol_offset={args.pol_offset}")
    shape = f"n={w.n};T={w.T};A={w.A};S={w.S}" if w is not None else \
        f"n={args.n_channels or 'default'};T={args.taps or 'default'};S={args.n_spectra or 'default'}"
    return f"config={args.config};{shape};bits={args.sample_bits};opts={'+'.join(opts)}"


def measured_peaks():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        d = json.loads(f.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi sampling of SM clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        # "under load" = samples at or above the median power
        med_p = statistics.median(power)
        load = [c for c, p in zip(sm, power) if p >= med_p] or sm
        return {"sm_mhz": statistics.median(load), "sm_max_mhz": max(smax), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(power)}


def oracle_timed(cfg: int, n_spectra: int, repeats: int = 1):
    """Time the oracle as it stands on a bounded sample (first n_spectra spectra of every stream)."""
    import oracle
    import synth_inputs as si
    w = si.make_workload(cfg, n_spectra=n_spectra)
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        oracle.process(w.packed, w.A, w.n, w.T, w.P, w.weights, w.S, coarse=w.coarse, fine_delay=w.fine_delay,
                       phase=w.phase, gains=w.gains, want_Y=False)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return w, best, oracle.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    n_sample = 64
    import oracle
    import synth_inputs as si
    w = si.make_workload(args.config, n_spectra=n_sample)
    def step():
        oracle.process(w.packed, w.A, w.n, w.T, w.P, w.weights, w.S, coarse=w.coarse, fine_delay=w.fine_delay,
                       phase=w.phase, gains=w.gains, want_Y=False)
    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / args.steps
    units = w.A * w.S * w.N
    value = units / dt / 1e9
    cores = oracle.num_threads()
    sample = f"first {n_sample} spectra of every stream of config {args.config} per step (float64 oracle, OpenMP)"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config{args.config}: {w.A} antennas x 2 pols, n={w.n}, T={w.T}, bounded sample",
                   "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--n-channels", type=int, default=None, help="sweep point for config 5")
    ap.add_argument("--n-spectra", type=int, default=None, help="shrink the batch (debugging only)")
    ap.add_argument("--sample-bits", type=int, default=10, help="input sample width (bit-depth sweep of PAPER.md:273-279)")
    ap.add_argument("--taps", type=int, default=None, help="override T (tap sweep of PAPER.md:235-249; 2, 4, 8, 16, 32)")
    ap.add_argument("--pol-offset", type=int, default=0,
                    help="add this many samples to the coarse delay of pol 1 of every antenna (PAPER.md:117: the two "
                         "polarisations may have different delays): measures the kernels an unequal-pol engine runs")
    ap.add_argument("--chunk-spectra", type=int, default=None)
    ap.add_argument("--fir-rows", type=int, default=None)
    ap.add_argument("--opt", action="append", default=[], help="library option key=value (fengine_set_option), repeatable")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--csrc-hash", action="store_true", help="print the kernel-source hash that profiles/roofline_traffic.csv is stamped with")
    args = ap.parse_args()
    if args.csrc_hash:
        print(csrc_hash())
        return 0
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import paper_2303_09886_b200 as fb
    import synth_inputs as si

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    fb.lib()                                             # fail loudly if the CUDA library is missing
    # Streams are independent: every rank runs the full configuration on its own antennas
    # (weak scaling, no data-path collective).  Different seed per rank = different antennas.
    w = si.make_workload(args.config, n_spectra=args.n_spectra, n_channels=args.n_channels, seed=rank, taps=args.taps, bits=args.sample_bits)
    fe = fb.FEngine(w.n, w.T, w.P, w.weights, n_antennas=w.A)
    if args.pol_offset:
        w.coarse = w.coarse.copy()
        w.coarse[:, 1] += args.pol_offset
    fe.set_coarse_delays(w.coarse)
    fe.set_fine_delays(w.fine_delay, w.phase)
    fe.set_gains(w.gains)
    if args.sample_bits != 10:
        fe.set_option("sample_bits", args.sample_bits)
    if args.chunk_spectra is not None:
        fe.set_option("chunk_spectra", args.chunk_spectra)
    if args.fir_rows is not None:
        fe.set_option("fir_rows", args.fir_rows)
    for kv in args.opt:
        k, v = kv.split("=")
        fe.set_option(k, int(v))

    host_in = torch.from_numpy(w.packed.reshape(-1))
    in_bytes, out_shape = host_in.numel(), fe.output_shape(w.S)
    out_bytes = int(np.prod(out_shape))
    # rotate over buffer sets so that the footprint of consecutive steps exceeds the 126 MB L2
    n_sets = max(2, int(np.ceil(1.5e9 / (in_bytes + out_bytes)))) if (in_bytes + out_bytes) < 1.0e9 else 2
    d_in = [host_in.cuda() for _ in range(n_sets)]
    d_out = [torch.empty(out_shape, dtype=torch.int8, device="cuda") for _ in range(n_sets)]
    units_per_step = w.A * w.S * w.N                    # dual-pol sample instants per step per rank

    def step(i):
        fe.process(d_in[i % n_sets], d_out[i % n_sets], w.S)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(max(args.warmup, 3)):
        step(i)
    barrier()
    sampler = ClockSampler(local_rank)
    time.sleep(0.15)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for i in range(args.steps):
        step(i)
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)                         # the contract's number: exactly K steps, nothing else in between
    # per-step distribution (median and spread) from a second pass with one event per step boundary,
    # recorded on the stream the kernels are launched on; kept out of the bracket above because an event record
    # costs a few microseconds, which the launch-bound config 1 would notice
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    marks[0].record()
    for i in range(args.steps):
        step(i)
        marks[i + 1].record()
    torch.cuda.synchronize()
    per_step = sorted(marks[i].elapsed_time(marks[i + 1]) for i in range(args.steps))
    def pct(q):
        return per_step[min(len(per_step) - 1, int(q * len(per_step)))]
    step_stats = {"median": statistics.median(per_step), "p10": pct(0.10), "p90": pct(0.90), "min": per_step[0],
                  "max": per_step[-1], "n": len(per_step)}
    launches = fe.last_launch_count() * args.steps
    # keep the GPU busy a little longer so the clock sampler sees enough loaded samples
    t_end = time.time() + 0.6
    i = 0
    while time.time() < t_end:
        step(i); i += 1
        if i % 8 == 0:
            torch.cuda.synchronize()
    torch.cuda.synchronize()
    clocks = sampler.stop()

    from paper_2303_09886_b200 import sharding
    ms_total = sharding.max_over_ranks(ms_total, dist if world > 1 else None, device="cuda")
    ms_per_step = ms_total / args.steps
    value = sharding.aggregate_rate(units_per_step, world, ms_per_step * 1e-3) / 1e9

    # ---- per-kernel durations (CUDA events recorded by the library on the launching stream) ----
    fe.set_option("profile", 1)
    n_prof = min(args.steps, 50)
    for i in range(n_prof):
        step(i)
    torch.cuda.synchronize()
    fir_ms, fft_ms, n_fir, n_fft = fe.profile_read()
    fe.set_option("profile", 0)
    peak, peak_src = measured_peaks()
    fir_avg, fft_avg = fir_ms / max(n_fir, 1), fft_ms / max(n_fft, 1)
    launches_per_step = max(n_fir // max(n_prof, 1), 1)
    dom_name, dom_avg = ("fft_kernel", fft_avg) if fft_avg >= fir_avg else ("fir_kernel", fir_avg)
    alg_bytes_per_unit = 2.0 * (args.sample_bits / 8.0 + 1.0)      # 4.5 at 10 bits (ALG_BYTES_PER_DUALPOL_SAMPLE)
    alg_bytes_launch = alg_bytes_per_unit * units_per_step / launches_per_step
    achieved = alg_bytes_launch / (dom_avg * 1e-3) / 1e9 if dom_avg > 0 else 0.0
    step_gbs = alg_bytes_per_unit * units_per_step / (ms_per_step * 1e-3) / 1e9
    roofline = {
        "bound": "hbm", "kernel": dom_name, "achieved": achieved, "peak": peak, "unit": "GB/s",
        "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
        "algorithmic_bytes_per_launch": alg_bytes_launch,
        "kernel_ms": {"fir_kernel": fir_avg, "fft_kernel": fft_avg, "launches_per_step_each": launches_per_step},
        "step_achieved": step_gbs, "step_frac": step_gbs / peak,
        "note": "achieved = 4.5 B per dual-pol sample x samples per launch / dominant kernel's mean duration; "
                "step_frac is the same bytes over the whole step (the metric's % of HBM roofline)",
    }
    # The path is bound by the plain FP32 pipe before it is bound by HBM:
    # north-star accounting, FIR 2T flop + FFT 5 n log2(n) / N flop per real sample; an FMA is one lane-operation
    # (2 flop), the FFT's adds and multiplies are one lane-operation each.  Peak = the packed-FP32 issue rate the
    # library measures in this run (fengine_debug_fp32_rate; about 124 lane-ops/clk/SM, profiles/r1_fp32_rate.txt).
    lane_ops_per_real = w.T + 5.0 * w.n * np.log2(w.n) / w.N
    alu_peak = fb.fp32_rate()                            # measured now, on this device, at the clocks of the moment
    alu_achieved = lane_ops_per_real * w.P * units_per_step / (ms_per_step * 1e-3)
    roofline["alu"] = {"bound": "alu", "achieved": alu_achieved / 1e12, "peak": alu_peak / 1e12, "unit": "T lane-op/s",
                       "frac": alu_achieved / alu_peak, "lane_ops_per_real_sample": lane_ops_per_real,
                       "peak_source": "fengine_debug_fp32_rate in this run (packed FFMA2 loop on every SM)",
                       "note": "whole step against the measured FP32 issue rate; the slower of this and the HBM roofline "
                               "is the north star's roofline"}
    roofline["fused"] = bool(n_fir and fir_avg < 0.02 * max(fft_avg, 1e-9))
    if roofline["fused"]:
        roofline["kernel"] = dom_name = "fused_kernel"
    # DRAM bytes per launch come from a committed `ncu --set full` capture (a number taken under the profiler is never
    # a bench value, and ncu cannot run inside this timed program).  The CSV names the sha256 of the kernel sources it
    # was taken from; when the sources have changed since, the figures are withheld (null) instead of going stale.
    prof = ROOT / "profiles" / "roofline_traffic.csv"
    roofline["traffic_step"] = None
    if prof.exists():
        rows, src_hash, src_workload = {}, None, None
        for ln in prof.read_text().splitlines():
            if ln.startswith("# csrc_sha256="):
                src_hash = ln.split("=", 1)[1].strip()
            if ln.startswith("# workload="):
                src_workload = ln.split("=", 1)[1].strip()
            parts = ln.split(",")
            if len(parts) == 2 and parts[1].isdigit():
                rows[parts[0]] = int(parts[1])
        roofline["traffic_workload"] = workload_stamp(args, w)
        if src_workload != roofline["traffic_workload"]:
            roofline["traffic_source"] = (f"withheld: the committed ncu capture is of another workload or option set "
                                          f"({src_workload}; profiles/roofline_traffic.csv)")
        elif src_hash == csrc_hash():
            roofline["traffic"] = rows.get(dom_name)
            names = ["fused_kernel"] if roofline["fused"] else ["fir_kernel", "fft_kernel"]
            if all(nm in rows for nm in names):
                roofline["traffic_step"] = sum(rows[nm] for nm in names)
            roofline["traffic_source"] = f"profiles/roofline_traffic.csv (ncu capture of these sources, sha256 {src_hash[:12]})"
        else:
            roofline["traffic_source"] = "withheld: csrc/ has changed since the committed ncu capture (profiles/roofline_traffic.csv)"

    # ---- end to end through fengine_process_host: pinned host buffers, H2D + path + D2H per step ----
    e2e = None
    if not args.no_e2e:
        pin_in = host_in.pin_memory()
        pin_out = torch.empty(out_shape, dtype=torch.int8).pin_memory()
        k_e2e = max(3, min(args.steps, 10))
        for _ in range(2):
            fe.process_host(pin_in, pin_out, w.S)
        barrier()
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            fe.process_host(pin_in, pin_out, w.S)      # synchronous: returns after the D2H copy completed
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        tt = torch.tensor([dt], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        dt = float(tt.item())
        e2e = {"value": world * units_per_step * k_e2e / dt / 1e9, "unit": UNIT, "h2d_bytes_per_step": int(in_bytes),
               "d2h_bytes_per_step": int(out_bytes), "steps": k_e2e, "checksum": int(pin_out.view(-1)[::4099].to(torch.int32).sum())}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and args.sample_bits == 10:
        import oracle
        t0 = time.perf_counter()
        oracle.process(w.packed, w.A, w.n, w.T, w.P, w.weights, w.S, coarse=w.coarse, fine_delay=w.fine_delay,
                       phase=w.phase, gains=w.gains, want_Y=False)
        dt = time.perf_counter() - t0
        cores = oracle.num_threads()
        cpu_baseline = {"value": w.A * w.S * w.N / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"one full batch of config {args.config} ({w.A * w.P * w.L / 1e6:.1f} M real samples, "
                                  f"all {w.S} spectra of every stream), {dt:.2f} s wall = {dt * cores:.0f} core-seconds"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "ms_per_step_stats": step_stats, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"config{args.config}: {w.A} antennas x {w.P} pols per GPU, n={w.n}, T={w.T}, "
                                   f"{w.L} samples per pol per step, S={w.S} spectra"
                                   + (f", pol 1 delayed by {args.pol_offset} more samples" if args.pol_offset else ""),
                       "path": fe.path(),
                       "l2_hygiene": f"inputs larger than L2: {n_sets} rotating buffer sets, "
                                     f"{(in_bytes + out_bytes) / 1e6:.0f} MB touched per step",
                       "parallelism": f"antennas sharded over {world} GPU(s), no collective"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "cpu_baseline": cpu_baseline,
            "pct_of_hbm_roofline": 100.0 * step_gbs / peak,
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
