#!/usr/bin/env python
"""bench.py -- SPIIR filter-sample updates/s on one B200 (BASELINE.json metric), with roofline,
end-to-end, secondary legs and CPU-oracle legs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference|paper_design]

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
  legs      : (default run only) the other driver-visible numbers, each timed the same way for a few
              milliseconds: configs[4], configs[3] (roofline counts the FIR FMAs), configs[0], the
              configs[2] sweep ends (L = 1 and 32; streamed 256-sample blocks and one bulk call of
              16384 samples), the exported x2 stages alone (HBM and FP32 fractions), and the paper's
              own kernel design on configs[1] (spiir_pd_filter).
  cpu_baseline : the float64 oracle, as it stands, on this box's host cores, on a bounded sample,
              timed in a fresh subprocess (no CUDA / NVML threads beside it): all cores and one thread.
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
HBM_FALLBACK_GBS = 7700.0       # B200_PROFILING.md nominal figure, used only when MEASURED_PEAKS.json is absent
# dram__bytes_read.sum + dram__bytes_write.sum of ONE spiir_filter_kernel launch, copied from the committed
# `ncu --set full` captures named in TRAFFIC_SOURCE; per launch, like roofline.achieved.  Not measured by this run.
NCU_DRAM_TRAFFIC = {"cfg1_many_filter_1024x256": 7.425536e6 + 0.019456e6,
                    "cfg4_full_bank_2x16384x256": 235.016960e6 + 546.211072e6}
TRAFFIC_SOURCE = ("constant from the ncu --set full capture in profiles/r2_summary.md, not measured by this run; "
                  "configs[1]: coefficients, delays and state once per block; the 33.5 MB SNR block is still in the "
                  "126 MB L2 when the kernel ends and is evicted by the flush outside the events")


def _dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def load_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


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


def make_plan(sp, w, flags=0, time_chunks=0, impl="ours", block=None):
    block = block or w.block
    if impl == "paper_design":
        if len(w.banks) != 1 or w.n_streams != 1:
            raise ValueError("--impl paper_design covers the single-rate, single-stream configs (0, 1, 2)")
        b = w.banks[0]
        plan = sp.PaperDesignPlan(b.a1, b.b0, b.delays, max_block=block)
        return plan, 3                                  # window staging, filter kernel, history carry (+ one memset node)
    if len(w.banks) == 1:
        b = w.banks[0]
        plan = sp.Plan(b.a1, b.b0, b.delays, b.rate_hz, n_streams=w.n_streams, max_block=block, flags=flags,
                       time_chunks=time_chunks)
        launches = plan.launch_info(block)["launches"]
    else:
        plan = sp.MultiratePlan([(b.a1, b.b0, b.delays) for b in w.banks], [b.rate_hz for b in w.banks],
                                n_streams=w.n_streams, max_block=block)
        launches = plan.launches(block)
    return plan, launches


def fir_fma_per_block(w, n_taps_down=192, n_taps_up=192):
    """FIR multiply-adds of one multirate block: every up-stage output is a complex sample =
    n_taps_up/2 taps x (re, im) = n_taps_up FMAs, for every (stream, template); every down-stage output is
    n_taps_down FMAs, once per stream."""
    H = len(w.banks)
    if H == 1:
        return 0
    up_out = sum(w.block >> h for h in range(H - 1))           # outputs per row over all up stages (4096 + ... + 128)
    down_out = sum(w.block >> h for h in range(1, H))
    return w.n_streams * (w.n_templates * up_out * n_taps_up + down_out * n_taps_down)


# -------------------------------------------------------------------------------------------------
# CPU legs (the oracle).  They run in a process that has no CUDA context, no NVML sampler and no torch
# thread pool beside the OpenMP team: `--impl reference` is such a process itself; the GPU arm spawns one.
# -------------------------------------------------------------------------------------------------
def cpu_model() -> str:
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.lower().startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def usable_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def oracle_env(threads: int) -> dict:
    env = dict(os.environ)
    env.update({"OMP_NUM_THREADS": str(threads), "OMP_PROC_BIND": "close", "OMP_PLACES": "cores", "OMP_DYNAMIC": "false",
                "CUDA_VISIBLE_DEVICES": ""})
    return env


def oracle_sample(w, budget_updates: float):
    """Bounded sample of the workload for the CPU legs: first T_s templates x n_b consecutive blocks
    (the strain generator continues past the config's block count, so n_b may exceed it)."""
    per_template_block = w.updates_per_block() / w.n_templates
    T_s = int(min(w.n_templates, max(8, budget_updates // (2 * per_template_block))))
    n_b = int(max(1, min(256, budget_updates // (T_s * per_template_block))))
    return T_s, n_b


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


def calibrated_oracle_sample(w, seconds: float):
    """Pick a sample that keeps the oracle busy for about `seconds` on this box's cores."""
    T0 = min(w.n_templates, 64)
    run_oracle(w, T0, 1)                                  # page the library and the inputs in
    rate, _, _ = run_oracle(w, T0, 1)
    return oracle_sample(w, rate * seconds)


def cpu_leg_main(args):
    """Child process of the GPU arm: one oracle timing with the thread count given by OMP_NUM_THREADS."""
    w = make_workload(args.config, 0, args.filters)
    T_s, n_b = calibrated_oracle_sample(w, args.cpu_seconds)
    v, dt, cores = run_oracle(w, T_s, n_b)
    print(json.dumps({"value": v, "seconds": dt, "cores": cores,
                      "sample": f"first {T_s} of {w.n_templates} templates x {n_b} block(s) of {w.block} samples"}), flush=True)
    return 0


def cpu_leg_subprocess(cfg: int, filters: int, seconds: float, threads: int):
    cmd = [sys.executable, os.path.abspath(__file__), "--cpu-leg", "--config", str(cfg), "--filters", str(filters),
           "--cpu-seconds", str(seconds)]
    out = subprocess.run(cmd, env=oracle_env(threads), capture_output=True, text=True, timeout=600)
    for ln in reversed(out.stdout.strip().splitlines()):
        if ln.startswith("{"):
            return json.loads(ln)
    raise RuntimeError("cpu leg failed: " + out.stderr[-400:])


def cpu_baseline(cfg: int, filters: int, seconds: float):
    cores = usable_cores()
    allc = cpu_leg_subprocess(cfg, filters, seconds, cores)
    one = cpu_leg_subprocess(cfg, filters, max(3.0, seconds / 3.0), 1)
    return {"value": allc["value"], "unit": UNIT, "cores": allc["cores"], "kind": "oracle", "seconds": allc["seconds"],
            "sample": allc["sample"], "single_thread": {"value": one["value"], "seconds": one["seconds"], "sample": one["sample"]},
            "cpu_model": cpu_model(), "how": "fresh subprocess, no CUDA context, OMP_PROC_BIND=close"}


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
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "cpu_model": cpu_model()},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# -------------------------------------------------------------------------------------------------
# Device timing
# -------------------------------------------------------------------------------------------------
class DeviceTimer:
    """K steps, each bracketed by CUDA events on the launching stream, an L2 flush (256 MiB write) between
    steps outside the events."""

    def __init__(self):
        import torch
        self.torch = torch
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
        self.stream = torch.cuda.current_stream()

    def run(self, step, steps: int, warmup: int, first: int = 0):
        torch = self.torch
        for i in range(warmup):
            step(first + i)
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        t0 = time.perf_counter()
        for i in range(steps):
            self.flush.fill_(i & 0xFF)
            ev[i][0].record(self.stream)
            step(first + warmup + i)
            ev[i][1].record(self.stream)
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        return np.array([a.elapsed_time(b) for a, b in ev]), wall


def graph_steps(torch, plan, x_dev, out, mode: str):
    """One CUDA graph per resident strain block (the library keeps every ping-pong phase on the device, so a
    captured call can be replayed for each block of the stream); eager launches if capture fails."""
    plan.filter(x_dev[0], out)                      # first call outside any capture (kernel attributes)
    torch.cuda.synchronize()
    graphs = None
    if mode != "off":
        try:
            graphs = []
            for xb in x_dev:
                g = torch.cuda.CUDAGraph()
                # thread_local: CUDA calls of other threads (NCCL watchdog, clock sampler) must not invalidate the capture
                with torch.cuda.graph(g, capture_error_mode="thread_local"):
                    plan.filter(xb, out)
                graphs.append(g)
        except Exception as exc:                     # pragma: no cover - depends on the driver
            if mode == "on":
                raise
            print(f"bench.py: CUDA graph capture failed ({exc}); eager launches", file=sys.stderr)
            graphs = None
    plan.reset()
    torch.cuda.synchronize()
    nblk = len(x_dev)
    if graphs is not None:
        return (lambda i: graphs[i % nblk].replay()), True
    return (lambda i: plan.filter(x_dev[i % nblk], out)), False


def fp32_peak_tflops(props, sm_max_mhz):
    return props.multi_processor_count * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12


def filter_leg(sp, timer, cfg: int, steps: int, warmup: int, peak_tflops: float, filters: int = 0, impl: str = "ours",
               bulk_blocks: int = 0, graph: str = "auto"):
    """One secondary leg: configs[cfg] (or its bulk shape: bulk_blocks blocks in ONE call) timed like the main leg."""
    import torch
    w = make_workload(cfg, 0, filters)
    n = w.block * (bulk_blocks or 1)
    plan, launches = make_plan(sp, w, impl=impl, block=n)
    nblk = 2 if bulk_blocks else min(w.n_blocks, 8)
    if bulk_blocks:
        xs = [np.concatenate([w.strain(k * bulk_blocks + i) for i in range(bulk_blocks)], -1) for k in range(nblk)]
    else:
        xs = [w.strain(i) for i in range(nblk)]
    x_dev = [torch.from_numpy(x).cuda() for x in xs]
    out = torch.empty((w.n_streams, w.n_templates, n), dtype=torch.complex64, device="cuda")
    step, graphed = graph_steps(torch, plan, x_dev, out, graph)
    ms, _ = timer.run(step, steps, warmup)
    upd = w.updates_per_block() * (bulk_blocks or 1)
    t = float(ms.mean()) * 1e-3
    fir = fir_fma_per_block(w)
    flop = FLOP_PER_UPDATE * upd + 2 * fir
    snr_bytes = w.n_streams * w.n_templates * n * 8
    leg = {"workload": w.name + (f"_bulk{n}" if bulk_blocks else ""), "impl": impl, "ms_per_step": t * 1e3, "steps": steps,
           "value": upd / t, "unit": UNIT, "launches_per_step": launches, "graph": graphed,
           "roofline": {"bound": "alu", "achieved": flop / t / 1e12, "peak": peak_tflops, "unit": "TFLOP/s",
                        "frac": flop / t / 1e12 / peak_tflops},
           "snr_writeback_gbs": snr_bytes / t / 1e9}
    if fir:
        leg["roofline"]["flop"] = {"filter_updates_x12": FLOP_PER_UPDATE * upd, "fir_fma_x2": 2 * fir}
    plan.close()
    del plan, out, x_dev
    torch.cuda.empty_cache()
    return leg


def resample_leg(sp, timer, direction: str, taps: int, rows: int, steps: int, warmup: int, hbm_peak: float, fma_peak: float):
    """The exported x2 stage alone on a batch large enough to leave the launch-bound regime (rows x 2048 -> 4096 up with
    accumulate, or rows x 4096 -> 2048 down).  Both rooflines DESIGN.md discusses: HBM (algorithmic bytes per output) and FP32."""
    import torch
    up = direction == "up"
    n_in = 2048 if up else 4096
    r = sp.Resampler("up" if up else "down", rows, max_block=n_in, n_taps=taps)
    if up:
        v = torch.randn(rows, n_in, dtype=torch.complex64, device="cuda")
        out = torch.zeros(rows, 2 * n_in, dtype=torch.complex64, device="cuda")
        call = lambda i: r.up(v, out, accumulate=True)
        n_out, bytes_per_out, fma_per_out = rows * 2 * n_in, 20.0, taps            # 4 in + 8 read + 8 written; taps/2 x (re, im)
    else:
        u = torch.randn(rows, n_in, dtype=torch.float32, device="cuda")
        out = torch.zeros(rows, n_in // 2, dtype=torch.float32, device="cuda")
        call = lambda i: r.down(u, out)
        n_out, bytes_per_out, fma_per_out = rows * n_in // 2, 12.0, taps           # 8 in + 4 written; one FMA per tap
    ms, _ = timer.run(call, steps, max(3, warmup))
    t = float(ms.mean()) * 1e-3
    gbs = n_out * bytes_per_out / t / 1e9
    leg = {"workload": f"resample_{direction}_{rows}x{n_in}_{taps}taps", "ms_per_step": t * 1e3, "steps": steps,
           "value": n_out / t, "unit": "output samples/s",
           "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                        "bytes_per_output": bytes_per_out},
           "roofline_alu": {"bound": "alu", "achieved": n_out * fma_per_out * 2 / t / 1e12, "peak": 2 * fma_peak / 1e12,
                            "unit": "TFLOP/s", "frac": n_out * fma_per_out / t / fma_peak, "fma_per_output": fma_per_out}}
    if up and taps in (192, 32):
        # this stage runs on the tensor cores (spiir_up2_tc_kernel): the FP32 figure is the CUDA-core rate the same useful
        # arithmetic would need, a fraction above 1 means CUDA cores could not do it in this time
        leg["roofline_alu"]["note"] = ("executed by tcgen05.mma (TF32 + two bf16 correction products), not by FP32 FMAs: "
                                       "useful FIR flops against the CUDA-core FP32 peak, for comparison with the CUDA-core kernel")
        leg["kernel"] = "spiir_up2_tc_kernel"
    r.close()
    del r, out
    torch.cuda.empty_cache()
    return leg


def secondary_legs(sp, timer, peak_tflops, hbm_peak, fma_peak, warmup):
    legs = {}

    def add(name, fn):
        try:
            legs[name] = fn()
        except Exception as exc:                      # a failed leg must not take the headline line down with it
            legs[name] = {"error": f"{type(exc).__name__}: {exc}"[:300]}

    add("cfg4", lambda: filter_leg(sp, timer, 4, 10, 3, peak_tflops))
    add("cfg3", lambda: filter_leg(sp, timer, 3, 50, warmup, peak_tflops))
    add("cfg0", lambda: filter_leg(sp, timer, 0, 50, warmup, peak_tflops))
    for L in (1, 32):
        add(f"cfg2_L{L}_streamed", lambda L=L: filter_leg(sp, timer, 2, 100, warmup, peak_tflops, filters=L))
        add(f"cfg2_L{L}_bulk", lambda L=L: filter_leg(sp, timer, 2, 20, 3, peak_tflops, filters=L, bulk_blocks=64))
    add("resample_up_192", lambda: resample_leg(sp, timer, "up", 192, 16384, 20, 3, hbm_peak, fma_peak))
    add("resample_down_192", lambda: resample_leg(sp, timer, "down", 192, 16384, 20, 3, hbm_peak, fma_peak))
    add("resample_up_32", lambda: resample_leg(sp, timer, "up", 32, 16384, 20, 3, hbm_peak, fma_peak))
    add("paper_design_cfg1", lambda: filter_leg(sp, timer, 1, 10, 3, peak_tflops, impl="paper_design"))
    for L in (1, 32):
        key = f"cfg2_L{L}_bulk"
        if "error" not in legs.get(key, {"error": 1}):
            # L <= 4 is bound by the complex64 SNR writeback (8 B per template-sample)
            legs[key]["roofline_hbm"] = {"bound": "hbm", "achieved": legs[key]["snr_writeback_gbs"], "peak": hbm_peak,
                                         "unit": "GB/s", "frac": legs[key]["snr_writeback_gbs"] / hbm_peak}
    return legs


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
    bulk = args.bulk if args.config == 2 else 0
    n = w.block * (bulk or 1)
    plan, launches = make_plan(sp, w, args.plan_flags, args.time_chunks, impl=args.impl, block=n)
    S, T = w.n_streams, w.n_templates
    upd = w.updates_per_block() * (bulk or 1)
    nblk = 2 if bulk else min(w.n_blocks, 16)
    if bulk:
        strains = [np.concatenate([w.strain(k * bulk + i) for i in range(bulk)], -1) for k in range(nblk)]
    else:
        strains = [w.strain(i) for i in range(nblk)]
    x_host = [torch.from_numpy(x).pin_memory() for x in strains]
    x_dev = [x.cuda() for x in x_host]
    out = torch.empty((S, T, n), dtype=torch.complex64, device="cuda")
    timer = DeviceTimer()
    stream = timer.stream

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    step, graphed = graph_steps(torch, plan, x_dev, out, args.graph)

    # ---- device-resident leg -------------------------------------------------------------------
    for i in range(args.warmup):
        step(i)
    barrier()
    sampler = ClockSampler(local_rank); sampler.start()
    step_ms, t_wall = timer.run(step, args.steps, 0, first=args.warmup)
    barrier()
    clocks = sampler.stop()
    tot_ms = max_over_ranks(float(step_ms.sum()), world, "cuda")
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
    if graphed:
        try:
            e2e_graphs = []
            for b in range(2):
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, capture_error_mode="thread_local"):
                    plan.filter(xin[b], out2[b])
                e2e_graphs.append(g)
        except Exception:                            # pragma: no cover
            e2e_graphs = None

    def e2e_steps(k, first):
        for i in range(k):
            b = i & 1
            stream.wait_event(freed[b])                               # out2[b] was drained to the host
            xin[b].copy_(x_host[(first + i) % nblk].reshape(S, n), non_blocking=True)   # H2D of this step's input
            if e2e_graphs is not None:
                e2e_graphs[b].replay()
            else:
                plan.filter(xin[b], out2[b])
            done[b].record(stream)
            with torch.cuda.stream(copy_stream):
                copy_stream.wait_event(done[b])
                z_host[b].copy_(out2[b].reshape(S, T, n), non_blocking=True)           # D2H of this step's result
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
    e2e_ms = max_over_ranks(e0.elapsed_time(e1), world, "cuda")
    e2e_value = upd * world * args.steps / (e2e_ms * 1e-3)
    del out2, z_host, xin

    if rank == 0:
        props = torch.cuda.get_device_properties(local_rank)
        peaks = load_peaks()
        sm_max_mhz = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
        hbm_peak = float(peaks.get("hbm_gbs") or HBM_FALLBACK_GBS)
        peak_tflops = fp32_peak_tflops(props, sm_max_mhz)
        fma_peak = props.multi_processor_count * FP32_LANES_PER_SM * sm_max_mhz * 1e6       # FMA lane-ops per second
        fir = fir_fma_per_block(w)
        flop = FLOP_PER_UPDATE * upd + 2 * fir
        achieved = flop / (ms_per_step * 1e-3) / 1e12
        kernel = {"ours": "spiir_filter_kernel", "paper_design": "spiir_pd_block_kernel (the paper's own design, comparison only)"}[args.impl]
        roofline = {"bound": "alu", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                    "frac": achieved / peak_tflops, "traffic": NCU_DRAM_TRAFFIC.get(w.name) if args.impl == "ours" and not bulk else None,
                    "traffic_note": TRAFFIC_SOURCE,
                    "kernel": kernel if len(w.banks) == 1 else "whole multirate step: spiir_filter_kernel banks + down chain + up cascade",
                    "peak_source": f"derived: {props.multi_processor_count} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 flop x "
                                   f"{sm_max_mhz:.0f} MHz (clocks.max.sm, MEASURED_PEAKS.json); 12 flop per update (PAPER.md:88)"
                                   + ("; FIR stages counted at 2 flop per tap-FMA" if fir else "")}
        if fir:
            roofline["flop"] = {"filter_updates_x12": FLOP_PER_UPDATE * upd, "fir_fma_x2": 2 * fir}
        # FMA-pipe view: an update needs 8 FP32 lane-ops (4 packed FFMA2-class instructions); the pipe peak is
        # SMs x 128 lane-ops per clock, so pipe utilisation = (8 x updates + FIR FMAs) / s / (SMs * 128 * clock)
        try:
            roofline["peak_measured_ffma_loop"] = sp.spiir_probe_fp32_peak()      # TFLOP/s of a register-only FFMA loop
            roofline["frac_of_measured"] = achieved / roofline["peak_measured_ffma_loop"]
        except Exception:
            pass
        roofline["fma_pipe_frac"] = (8.0 * upd + fir) / (ms_per_step * 1e-3) / fma_peak
        snr_bytes = S * T * n * 8
        legs = None
        if args.legs == "on" or (args.legs == "auto" and args.config == 1 and args.impl == "ours" and world == 1 and not bulk):
            plan.close()
            del out, x_dev
            torch.cuda.empty_cache()
            legs = secondary_legs(sp, timer, peak_tflops, hbm_peak, fma_peak, min(args.warmup, 8))
        cpu = None
        if not args.no_cpu:
            try:
                cpu = cpu_baseline(args.config, args.filters, args.cpu_seconds)
            except Exception as exc:
                cpu = {"error": f"{type(exc).__name__}: {exc}"[:300]}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": w.name + (f"_bulk{n}" if bulk else ""), "templates_per_gpu": T,
                           "filters_per_template": int(sum(b.a1.shape[1] for b in w.banks)),
                           "streams": S, "block_samples": n, "rate_hz": w.banks[0].rate_hz,
                           "updates_per_step_per_gpu": upd, "l2": "flushed between timed steps (256 MiB write)",
                           "launch": "one CUDA graph replay per step" if graphed else "eager launches",
                           "parallelism": f"template shards x{world}, no collective"},
                "pct_fp32_peak": 100.0 * achieved / peak_tflops,
                "data_seconds_per_wall_second": (n / w.banks[0].rate_hz) / (ms_per_step * 1e-3),
                "snr_writeback_gbs": snr_bytes / (ms_per_step * 1e-3) / 1e9,
                "step_ms_min_median_max": [float(step_ms.min()), float(np.median(step_ms)), float(step_ms.max())],
                "wall_ms_per_step_incl_flush": t_wall * 1e3 / args.steps,
                "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": S * n * 4, "d2h_bytes_per_step": snr_bytes,
                        "ms_per_step": e2e_ms / args.steps,
                        "note": "bound by the D2H copy of the SNR block over PCIe, not by the kernels"},
                "gpu_launches": launches * args.steps,
                "roofline": roofline,
                "cpu_baseline": cpu}
        if args.impl != "ours":
            line["impl"] = args.impl
        if legs is not None:
            line["legs"] = legs
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def bench_resample(args):
    """Standalone x2 stage: see resample_leg."""
    import torch
    import paper_1702_02256_b200 as sp
    sp.lib()
    torch.cuda.set_device(0)
    peaks = load_peaks()
    props = torch.cuda.get_device_properties(0)
    timer = DeviceTimer()
    sampler = ClockSampler(0); sampler.start()
    sm_max_mhz = float(peaks.get("sm_max_mhz") or 1965.0)
    fma_peak = props.multi_processor_count * FP32_LANES_PER_SM * sm_max_mhz * 1e6
    leg = resample_leg(sp, timer, args.resample, args.taps, args.rows, args.steps, args.warmup,
                       float(peaks.get("hbm_gbs") or HBM_FALLBACK_GBS), fma_peak)
    clocks = sampler.stop()
    line = {"metric": f"x2 resampler ({args.resample}) output samples/s", "value": leg["value"], "unit": "samples/s",
            "n_gpus": 1, "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": leg["ms_per_step"],
            "higher_is_better": True, "dtype": "f32", "data": "synthetic",
            "config": {"workload": leg["workload"], "rows": args.rows, "n_taps": args.taps,
                       "l2": "flushed between timed steps (256 MiB write)"},
            "clocks": clocks, "gpu_launches": args.steps, "roofline": leg["roofline_alu"], "roofline_hbm": leg["roofline"]}
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=16)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index (default 1: the metric's config)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference", "paper_design"],
                    help="reference: the float64 oracle on the host cores; paper_design: the paper's own (Maxwell) kernel "
                         "design restated for this GPU (spiir_pd_filter, comparison only)")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of one oracle sample")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--legs", default="auto", choices=["auto", "on", "off"],
                    help="secondary legs in the JSON line (auto: only in the default configs[1] run on one GPU)")
    ap.add_argument("--time-chunks", type=int, default=0, help="spiir_plan_opts.time_chunks (0 auto, 1 never chunk)")
    ap.add_argument("--filters", type=int, default=0, help="config 2 only: filters per template of the sweep point")
    ap.add_argument("--bulk", type=int, default=0, help="config 2 only: this many 256-sample blocks in ONE call (64: n = 16384)")
    ap.add_argument("--resample", default="", choices=["", "up", "down"],
                    help="time the exported x2 stage alone (rows x 2048 -> 4096 up+accumulate, or rows x 4096 -> 2048 down)")
    ap.add_argument("--rows", type=int, default=16384, help="rows of the --resample batch")
    ap.add_argument("--taps", type=int, default=192, choices=[32, 192, 384],
                    help="FIR length of the --resample stage (192: configs[3]; 32 / 384: the paper's own up / down filters, PAPER.md:88)")
    ap.add_argument("--graph", default="auto", choices=["auto", "on", "off"],
                    help="replay one captured CUDA graph per step (auto: fall back to eager launches if capture fails)")
    ap.add_argument("--plan-flags", type=int, default=0, help="spiir_plan_opts.flags (bit 0: skip the bank-conflict-avoiding permutation)")
    ap.add_argument("--cpu-leg", action="store_true", help=argparse.SUPPRESS)
    args = ap.parse_args()
    if args.cpu_leg:
        return cpu_leg_main(args)
    if args.warmup < 3 and args.impl != "reference":
        args.warmup = 3
    if args.resample:
        return bench_resample(args)
    if args.impl == "reference":
        return bench_reference(args)
    return bench_ours(args)


if __name__ == "__main__":
    if "--impl" in sys.argv and "reference" in sys.argv or "--cpu-leg" in sys.argv:
        # the oracle's OpenMP team: pinned, one thread per usable core, set before the library loads
        os.environ.setdefault("OMP_NUM_THREADS", str(usable_cores()))
        os.environ.setdefault("OMP_PROC_BIND", "close")
        os.environ.setdefault("OMP_PLACES", "cores")
        os.environ.setdefault("OMP_DYNAMIC", "false")
    sys.exit(main())
