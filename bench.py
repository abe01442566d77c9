#!/usr/bin/env python
"""bench.py -- SPIIR filter-sample updates/s on one B200 (BASELINE.json metric), with roofline,
end-to-end and CPU-oracle legs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference]

A "step" is one streamed block of the workload through the whole hot path (spiir_filter, or
spiir_mr_filter for config 3): for the default workload (BASELINE.json configs[1], the config the
metric is quoted on) that is 4096 samples x 1024 templates x 256 filters = 1.07e9 Eq.-7 updates,
with filter state and input history carried from the previous step.

Timed legs:
  value     : updates/s with the strain blocks resident in HBM; every step is bracketed by CUDA
              events on the launching stream; an L2 flush (256 MiB write) runs between steps,
              outside the events.
  e2e       : the same metric through the same public call with HOST buffers: every step copies
              its strain block from pinned host memory, filters, and copies the complex64 SNR
              block back to pinned host memory (double-buffered on a copy stream).
  roofline  : FP32 ALU bound: 12 flop per update / kernel time, against
              SMs x 128 lanes x 2 flop x clocks.max.sm (DESIGN.md derives it).
  cpu_baseline : the float64 oracle, as it stands, on this box's host cores, on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "SPIIR filter-sample updates/s (templates*filters*samples/s)"
UNIT = "updates/s"
FLOP_PER_UPDATE = 12
FP32_LANES_PER_SM = 128         # B200 SM: 4 sub-partitions x 32 FP32 lanes (guides/B300_MICROARCH.md)
# dram__bytes_read.sum + dram__bytes_write.sum of one spiir_filter_kernel launch, from the committed
# `ncu --set full` captures (profiles/r1c_summary.md); per launch, like roofline.achieved
NCU_DRAM_TRAFFIC = {"cfg1_many_filter_1024x256": 7.428352e6 + 0.137472e6,
                    "cfg4_full_bank_2x16384x256": 235.036672e6 + 556.152064e6}


def _dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self._halt = index, [], threading.Event()

    def _nvml_loop(self) -> bool:
        """Fast path: NVML through nvidia_ml_py (sub-millisecond samples).  False if NVML is unusable."""
        try:
            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            mx = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
        except Exception:
            return False
        bits = {"hw_slowdown": getattr(pynvml, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
                "hw_thermal_slowdown": getattr(pynvml, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                "sw_thermal_slowdown": getattr(pynvml, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
                "sw_power_cap": getattr(pynvml, "nvmlClocksThrottleReasonSwPowerCap", 0x4)}
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        while not self._halt.is_set():
            try:
                sm = pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)
                r = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                self.rows.append([str(sm), str(mx), "0"] + ["Active" if r & bits[n] else "Not Active" for n in names])
            except Exception:
                pass
            self._halt.wait(0.005)
        return True

    def run(self):
        if self._nvml_loop():
            return
        while not self._halt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([c.strip() for c in out.strip().split(",")])
            except Exception:
                pass
            self._halt.wait(0.1)

    def stop(self):
        self._halt.set()
        self.join(timeout=6)
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
                for nm, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


def max_over_ranks(value: float, world: int, device="cpu") -> float:
    """Timing rule for N > 1: every rank reports the slowest rank's device time (all_reduce MAX)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def make_workload(cfg: int, rank: int, n_filters: int = 0):
    """BASELINE.json configs[cfg]; rank r > 0 gets its own template shard (different seed stream)."""
    from paper_1702_02256_b200 import inputs
    w = inputs.config(cfg, n_filters=n_filters or None) if cfg == 2 else inputs.config(cfg)
    if rank:
        # independent template partition per rank (weak scaling, no data-path collective): reseed
        from dataclasses import replace
        banks = tuple(inputs.make_bank(tuple(w.seed_key) + (1000 + rank, h), b.a1.shape[0], b.a1.shape[1], b.rate_hz,
                                       0.5 if cfg == 2 else 0.9, 0.999 if cfg == 2 else 0.9999, int(b.delays.max()))
                      for h, b in enumerate(w.banks))
        w = replace(w, banks=banks)
    return w


def make_plan(sp, w, flags=0, time_chunks=0):
    if len(w.banks) == 1:
        b = w.banks[0]
        plan = sp.Plan(b.a1, b.b0, b.delays, b.rate_hz, n_streams=w.n_streams, max_block=w.block, flags=flags,
                       time_chunks=time_chunks)
        launches = plan.launch_info(w.block)["launches"]
    else:
        plan = sp.MultiratePlan([(b.a1, b.b0, b.delays) for b in w.banks], [b.rate_hz for b in w.banks],
                                n_streams=w.n_streams, max_block=w.block)
        launches = plan.launches(w.block)
    return plan, launches


def oracle_sample(w, budget_updates: float):
    """Bounded sample of the workload for the CPU legs: first T_s templates x n_b consecutive blocks
    (the strain generator continues past the config's block count, so n_b may exceed it)."""
    per_template_block = w.updates_per_block() / w.n_templates
    T_s = int(min(w.n_templates, max(8, budget_updates // (2 * per_template_block))))
    n_b = int(max(1, min(256, budget_updates // (T_s * per_template_block))))
    return T_s, n_b


def calibrated_oracle_sample(w, seconds: float):
    """Pick a sample that keeps the oracle busy for about `seconds` on this box's cores."""
    T0 = min(w.n_templates, 64)
    rate, _, _ = run_oracle(w, T0, 1)
    return oracle_sample(w, rate * seconds)


def run_oracle(w, T_s: int, n_b: int):
    """Times the oracle (float64, as it stands) on the first T_s templates for n_b blocks."""
    import oracle
    banks = [(b.a1[:T_s], b.b0[:T_s], b.delays[:T_s]) for b in w.banks]
    orc = oracle.FilterOracle(*banks[0], w.n_streams) if len(banks) == 1 else oracle.MultirateOracle(banks, w.n_streams)
    xs = [w.strain(i) for i in range(n_b)]
    t0 = time.perf_counter()
    for x in xs:
        orc.filter(x)
    dt = time.perf_counter() - t0
    upd = w.updates_per_block() / w.n_templates * T_s * n_b
    return upd / dt, dt, oracle.num_threads()


def bench_reference(args):
    rank, _, world = _dist_env()
    if rank != 0:
        return 0
    w = make_workload(args.config, 0, args.filters)
    # every step is a bounded sample; the whole --steps run stays within a few minutes of CPU time
    T_s, n_b = calibrated_oracle_sample(w, min(args.cpu_seconds, 150.0 / max(1, args.steps)))
    for _ in range(min(args.warmup, 1)):
        run_oracle(w, min(T_s, 16), 1)
    vals, times, cores = [], [], 1
    for _ in range(args.steps):
        v, dt, cores = run_oracle(w, T_s, n_b)
        vals.append(v); times.append(dt)
    value = float(np.sum([v * t for v, t in zip(vals, times)]) / np.sum(times))
    sample = f"first {T_s} of {w.n_templates} templates x {n_b} block(s) of {w.block} samples per step"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean(times) * 1e3),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def bench_ours(args):
    import torch
    import torch.distributed as dist
    rank, local_rank, world = _dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the SPIIR hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    import paper_1702_02256_b200 as sp
    sp.lib()

    w = make_workload(args.config, rank, args.filters)
    plan, launches = make_plan(sp, w, args.plan_flags, args.time_chunks)
    S, T, n = w.n_streams, w.n_templates, w.block
    upd = w.updates_per_block()
    nblk = min(w.n_blocks, 16)
    x_host = [torch.from_numpy(w.strain(i)).pin_memory() for i in range(nblk)]
    x_dev = [x.cuda() for x in x_host]
    out = torch.empty((S, T, n), dtype=torch.complex64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # One CUDA graph per resident strain block (the library keeps every ping-pong phase on the device, so
    # a captured call can be replayed for each block of the stream); eager launches if capture fails.
    def capture(xbuf, obuf):
        g = torch.cuda.CUDAGraph()
        # thread_local: CUDA calls of other threads (NCCL watchdog, clock sampler) must not invalidate the capture
        with torch.cuda.graph(g, capture_error_mode="thread_local"):
            plan.filter(xbuf, obuf)
        return g

    plan.filter(x_dev[0], out)                      # first call outside any capture (kernel attributes)
    torch.cuda.synchronize()
    graphs = None
    if args.graph != "off":
        try:
            graphs = [capture(x_dev[i], out) for i in range(nblk)]
        except Exception as exc:                     # pragma: no cover - depends on the driver
            if args.graph == "on":
                raise
            print(f"bench.py: CUDA graph capture failed ({exc}); eager launches", file=sys.stderr)
            graphs = None
        plan.reset()
        torch.cuda.synchronize()

    def step(i):
        if graphs is not None:
            graphs[i % nblk].replay()
        else:
            plan.filter(x_dev[i % nblk], out)

    # ---- device-resident leg -------------------------------------------------------------------
    for i in range(args.warmup):
        step(i)
    barrier()
    sampler = ClockSampler(local_rank); sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    t_wall0 = time.perf_counter()
    for i in range(args.steps):
        flush.fill_(i & 0xFF)                       # L2 flush between timed steps (outside the events)
        ev[i][0].record(stream)
        step(args.warmup + i)
        ev[i][1].record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    step_ms = np.array([a.elapsed_time(b) for a, b in ev])
    tot_ms = float(step_ms.sum())
    tot_ms = max_over_ranks(tot_ms, world, "cuda")
    ms_per_step = tot_ms / args.steps
    value = upd * world / (ms_per_step * 1e-3)

    # ---- end-to-end leg: pinned host -> device -> filter -> pinned host ----------------------------
    out2 = [torch.empty((S, T, n), dtype=torch.complex64, device="cuda") for _ in range(2)]
    z_host = [torch.empty((S, T, n), dtype=torch.complex64).pin_memory() for _ in range(2)]
    xin = [torch.empty((S, n), dtype=torch.float32, device="cuda") for _ in range(2)]
    copy_stream = torch.cuda.Stream()
    done = [torch.cuda.Event() for _ in range(2)]
    freed = [torch.cuda.Event() for _ in range(2)]

    e2e_graphs = None
    if graphs is not None:
        try:
            e2e_graphs = [capture(xin[b], out2[b]) for b in range(2)]
        except Exception:                            # pragma: no cover
            e2e_graphs = None

    def e2e_steps(k, first):
        for i in range(k):
            b = i & 1
            stream.wait_event(freed[b])                               # out2[b] was drained to the host
            xin[b].copy_(x_host[(first + i) % nblk], non_blocking=True)   # H2D of this step's input
            if e2e_graphs is not None:
                e2e_graphs[b].replay()
            else:
                plan.filter(xin[b], out2[b])
            done[b].record(stream)
            with torch.cuda.stream(copy_stream):
                copy_stream.wait_event(done[b])
                z_host[b].copy_(out2[b], non_blocking=True)           # D2H of this step's result
                freed[b].record(copy_stream)

    plan.reset()
    e2e_steps(max(3, min(args.warmup, 4)), 0)
    barrier(); copy_stream.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    e2e_steps(args.steps, 0)
    stream.wait_stream(copy_stream)
    e1.record(stream)
    barrier(); copy_stream.synchronize()
    e2e_ms = e0.elapsed_time(e1)
    e2e_ms = max_over_ranks(e2e_ms, world, "cuda")
    e2e_value = upd * world * args.steps / (e2e_ms * 1e-3)

    if rank == 0:
        props = torch.cuda.get_device_properties(local_rank)
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        sm_max_mhz = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
        peak_tflops = props.multi_processor_count * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
        achieved = FLOP_PER_UPDATE * upd / (ms_per_step * 1e-3) / 1e12
        roofline = {"bound": "alu", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                    "frac": achieved / peak_tflops, "traffic": NCU_DRAM_TRAFFIC.get(w.name),
                    "kernel": "spiir_filter_kernel" if len(w.banks) == 1 else "spiir_filter_kernel + resamplers (whole step)",
                    "peak_source": f"derived: {props.multi_processor_count} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 flop x "
                                   f"{sm_max_mhz:.0f} MHz (clocks.max.sm, MEASURED_PEAKS.json); 12 flop per update (PAPER.md:88)"}
        # FMA-pipe view: an update needs 8 FP32 lane-ops (4 packed FFMA2-class instructions); the pipe peak is
        # SMs x 128 lane-ops per clock, so pipe utilisation = updates/s * 8 / (SMs * 128 * clock)
        try:
            roofline["peak_measured_ffma_loop"] = sp.spiir_probe_fp32_peak()      # TFLOP/s of a register-only FFMA loop
            roofline["frac_of_measured"] = achieved / roofline["peak_measured_ffma_loop"]
        except Exception:
            pass
        roofline["fma_pipe_frac"] = (upd / (ms_per_step * 1e-3)) * 8.0 / (props.multi_processor_count * FP32_LANES_PER_SM * sm_max_mhz * 1e6)
        snr_bytes = S * T * n * 8
        cpu = None
        if not args.no_cpu:
            T_s, n_b = calibrated_oracle_sample(w, args.cpu_seconds)
            v, dt, cores = run_oracle(w, T_s, n_b)
            cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
                   "sample": f"first {T_s} of {T} templates x {n_b} block(s) of {n} samples"}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": w.name, "templates_per_gpu": T, "filters_per_template": int(sum(b.a1.shape[1] for b in w.banks)),
                           "streams": S, "block_samples": n, "rate_hz": w.banks[0].rate_hz,
                           "updates_per_step_per_gpu": upd, "l2": "flushed between timed steps (256 MiB write)",
                           "launch": "one CUDA graph replay per step" if graphs is not None else "eager launches",
                           "parallelism": f"template shards x{world}, no collective"},
                "pct_fp32_peak": 100.0 * achieved / peak_tflops,
                "data_seconds_per_wall_second": (n / w.banks[0].rate_hz) / (ms_per_step * 1e-3),
                "snr_writeback_gbs": snr_bytes / (ms_per_step * 1e-3) / 1e9,
                "step_ms_min_median_max": [float(step_ms.min()), float(np.median(step_ms)), float(step_ms.max())],
                "wall_ms_per_step_incl_flush": t_wall * 1e3 / args.steps,
                "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": S * n * 4, "d2h_bytes_per_step": snr_bytes,
                        "ms_per_step": e2e_ms / args.steps},
                "gpu_launches": launches * args.steps,
                "roofline": roofline,
                "cpu_baseline": cpu}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def bench_resample(args):
    """Standalone x2 stage (spiir_resample_up with accumulate / spiir_resample_down) on a batch large enough
    to leave the launch-bound regime: rows = 16384, 2048 -> 4096 (up) or 4096 -> 2048 (down), 192 taps.
    Reports both rooflines DESIGN.md discusses: HBM (algorithmic bytes per output) and FP32 FMA."""
    import torch
    import paper_1702_02256_b200 as sp
    sp.lib()
    torch.cuda.set_device(0)
    up = args.resample == "up"
    rows, n_in, taps = args.rows, (2048 if up else 4096), args.taps
    r = sp.Resampler("up" if up else "down", rows, max_block=n_in, n_taps=taps)
    if up:
        v = torch.randn(rows, n_in, dtype=torch.complex64, device="cuda")
        out = torch.zeros(rows, 2 * n_in, dtype=torch.complex64, device="cuda")
        call = lambda: r.up(v, out, accumulate=True)
        n_out, bytes_per_out, fma_per_out = rows * 2 * n_in, 20.0, taps            # 4 in + 8 read + 8 written; taps/2 x (re, im)
    else:
        u = torch.randn(rows, n_in, dtype=torch.float32, device="cuda")
        out = torch.zeros(rows, n_in // 2, dtype=torch.float32, device="cuda")
        call = lambda: r.down(u, out)
        n_out, bytes_per_out, fma_per_out = rows * n_in // 2, 12.0, taps           # 8 in + 4 written; one FMA per tap
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    for _ in range(max(3, args.warmup)):
        call()
    torch.cuda.synchronize()
    sampler = ClockSampler(0); sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for i in range(args.steps):
        flush.fill_(i & 0xFF)
        ev[i][0].record(stream); call(); ev[i][1].record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs") or 6542.7)
    props = torch.cuda.get_device_properties(0)
    sm_max_mhz = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    fma_peak = props.multi_processor_count * FP32_LANES_PER_SM * sm_max_mhz * 1e6           # FMA lane-ops per second
    gbs = n_out * bytes_per_out / (ms * 1e-3) / 1e9
    line = {"metric": f"x2 resampler ({args.resample}) output samples/s", "value": n_out / (ms * 1e-3), "unit": "samples/s",
            "n_gpus": 1, "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": ms, "higher_is_better": True,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"resample_{args.resample}_{rows}x{n_in}_{taps}taps", "rows": rows, "n_in": n_in, "n_taps": taps,
                       "l2": "flushed between timed steps (256 MiB write)"},
            "clocks": clocks, "gpu_launches": args.steps,
            "roofline": {"bound": "alu", "achieved": n_out * fma_per_out * 2 / (ms * 1e-3) / 1e12, "peak": 2 * fma_peak / 1e12,
                         "unit": "TFLOP/s", "frac": n_out * fma_per_out / (ms * 1e-3) / fma_peak, "traffic": None,
                         "kernel": f"spiir_up2_fir_kernel<{taps // 2}>" if up else f"spiir_down2_fir_kernel<{taps}>",
                         "note": f"{taps} FMA per output sample (DESIGN.md 5.2: 192 taps are FP32-bound, 32 taps HBM-bound)"},
            "roofline_hbm": {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                             "bytes_per_output": bytes_per_out}}
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=16)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index (default 1: the metric's config)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of one oracle sample")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--time-chunks", type=int, default=0, help="spiir_plan_opts.time_chunks (0 auto, 1 never chunk)")
    ap.add_argument("--filters", type=int, default=0, help="config 2 only: filters per template of the sweep point")
    ap.add_argument("--resample", default="", choices=["", "up", "down"],
                    help="time the exported x2 stage alone (rows x 2048 -> 4096 up+accumulate, or rows x 4096 -> 2048 down)")
    ap.add_argument("--rows", type=int, default=16384, help="rows of the --resample batch")
    ap.add_argument("--taps", type=int, default=192, choices=[32, 192],
                    help="FIR length of the --resample stage (192: configs[3]; 32: the paper's own up-filter, PAPER.md:88)")
    ap.add_argument("--graph", default="auto", choices=["auto", "on", "off"],
                    help="replay one captured CUDA graph per step (auto: fall back to eager launches if capture fails)")
    ap.add_argument("--plan-flags", type=int, default=0, help="spiir_plan_opts.flags (bit 0: skip the bank-conflict-avoiding permutation)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.resample:
        return bench_resample(args)
    if args.impl == "reference":
        return bench_reference(args)
    return bench_ours(args)


if __name__ == "__main__":
    sys.exit(main())
