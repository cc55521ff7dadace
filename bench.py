#!/usr/bin/env python
"""bench.py -- one JSON line for the hot path M = R (*) S + N of arXiv 2203.02479 on B200.

    python bench.py --gpus N --steps K --warmup W            # this repo's CUDA path (libwcsim.so through the C ABI)
    python bench.py --impl reference --steps K --warmup W    # the fp64 CPU oracle, as it stands, on the host cores

A "step" is one plane-event of BASELINE.json configs[1] (800 wires x 6000 ticks padded to 1024 x 8192, 100k depos,
binomial fluctuation on): clear S, raster + fluctuate + scatter-add, FFT-convolve with the response.  `value` is
depositions per second through that whole path (so ms_per_step is the "ms per plane-event" of BASELINE.json's
metric), inputs resident in HBM; `e2e` is the same through wcsim_simulate_host with pinned HOST buffers, the
host<->device copies inside the timed region.  L2 (126 MB) is flushed between timed steps by writing a 256 MB
buffer, outside the per-step CUDA-event pairs.  `roofline` is the dominant kernel's (the fluctuated raster: ALU bound),
with the FFT-convolve stage's HBM fractions under roofline.convolve; per-kernel durations come from a second pass of
the same K steps with CUDA-event pairs around every stage.  Multi-GPU: replicas only, one process per GPU.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC, UNIT = "depos_per_sec_plane_event", "depos/s"
FLUSH_BYTES = 256 << 20


def load_peaks():
    """Measured roofline denominators (driver-written MEASURED_PEAKS.json), else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            p = json.load(f)
        return {"hbm_gbs": float(p["hbm_gbs"]), "source": "measured (MEASURED_PEAKS.json)",
                "sm_max_mhz": float(p.get("sm_max_mhz", 1965.0))}
    except Exception:
        return {"hbm_gbs": 6650.0, "source": "fallback (B200_PROFILING.md)", "sm_max_mhz": 1965.0}


def stage_bytes(pl, direct, K=1):
    """Algorithmic HBM bytes of each convolution kernel for one plane-event; K impact positions
    per wire make the charge grid and the row spectra K times taller (reading A25)."""
    nw, nt, pw, pt = pl["n_wires"], pl["n_ticks"], pl["pad_w"], pl["pad_t"]
    nk = pt // 2 + 1
    grid, spec = nw * nt * 4, nw * nk * 8
    n_rw = pl["response"].shape[-2]
    resp = K * n_rw * nk * 8 if direct else pw * nk * 8  # Rt rows (direct) or Rhat (FFT wire mode)
    return {"rows_forward": K * (grid + spec), "cols": (K + 1) * spec + resp, "rows_inverse": spec + grid}


def nvml_index(local_rank):
    """NVML index of the rank's GPU: CUDA_VISIBLE_DEVICES may renumber devices; UUID / MIG entries or a list shorter than
    the rank fall back to the local rank (the sampler then reports what that device does, or 'unsampled')."""
    try:
        return int(os.environ["CUDA_VISIBLE_DEVICES"].split(",")[local_rank])
    except (KeyError, IndexError, ValueError):
        return local_rank


class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU while the timed region runs (NVML, in a thread)."""

    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
    NOTE = {"sw_power_cap": 0x4}

    def __init__(self, index, period=0.005):
        self.index, self.period = index, period
        self.mhz, self.reasons, self.max_mhz = [], 0, None
        self._stop = threading.Event()
        self._thread = None
        self._h = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._h = None

    def sample(self):
        if self._h is None:
            return
        try:
            self.mhz.append(float(self._nv.nvmlDeviceGetClockInfo(self._h, self._nv.NVML_CLOCK_SM)))
            try:
                r = self._nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
            except Exception:
                r = self._nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
            self.reasons |= int(r)
        except Exception:
            pass

    def _run(self):
        while not self._stop.is_set():
            self.sample()
            self._stop.wait(self.period)

    def start(self):
        self.sample()
        self._thread = threading.Thread(target=self._run, daemon=True)
        self._thread.start()

    def stop(self):
        self.sample()
        self._stop.set()
        if self._thread:
            self._thread.join()

    def summary(self):
        names = [n for n, bit in {**self.BAD, **self.NOTE}.items() if self.reasons & bit]
        if not self.mhz:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unsampled"], "samples": 0}
        return {"sm_mhz": statistics.median(self.mhz), "sm_max_mhz": self.max_mhz, "reasons": names,
                "samples": len(self.mhz)}


# --------------------------------------------------------------------------------------------------------------------
# this repo's arm
# --------------------------------------------------------------------------------------------------------------------
def run_ours(args):
    import numpy as np
    import torch
    from paper_2203_02479_b200 import binding as B, replicas, synth

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    rank, local_rank, world = replicas.env_world()
    if world != args.gpus and world > 1:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d" % (args.gpus, world))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    replicas.init("nccl")
    B.lib()  # fails loudly here if libwcsim.so cannot be built or loaded

    kw = {}
    if args.sigma_scale != 1.0:
        kw["sigma_scale"] = args.sigma_scale
    if args.shuffle:
        kw["shuffle"] = True  # the depo order as a sensitivity (generation order is the default)
    cfg = synth.config(args.config, **kw)
    pl = cfg["planes"][0]
    n_depos = int(pl["depos"]["t0"].shape[0])
    fluct = bool(cfg["fluctuate"]) and not args.no_fluct
    if fluct and args.fluct == "normal":
        fluct = 2
    mode = {"atomic": B.WCSIM_SCATTER_ATOMIC, "tiled": B.WCSIM_SCATTER_TILED, "fixed": B.WCSIM_SCATTER_FIXED}[args.scatter]
    stream = torch.cuda.current_stream()
    if args.impact > 1:
        # labelled variant (reading A25): K impact positions per wire, depos in units of pitch / K
        pl = dict(pl, depos=synth.to_impact_units(pl["depos"], args.impact),
                  response=synth.response_impact(args.impact, *pl["response"].shape))

    def make_plan(st):
        if args.impact > 1:
            return B.ImpactPlan(pl["n_wires"], pl["n_ticks"], pl["response"], pad_ticks=pl["pad_t"], nsigma=cfg["nsigma"],
                                scatter_mode=mode, stream=st)
        p_ = B.Plan(pl["n_wires"], pl["n_ticks"], pl["response"], pad=(pl["pad_w"], pl["pad_t"]), nsigma=cfg["nsigma"],
                    scatter_mode=mode, stream=st)
        p_.set_wire_mode({"auto": B.WCSIM_WIRES_AUTO, "fft": B.WCSIM_WIRES_FFT, "direct": B.WCSIM_WIRES_DIRECT}[args.wires])
        return p_

    plan = make_plan(stream)
    d = {k: torch.from_numpy(v).to(dev) for k, v in pl["depos"].items()}
    flush = torch.empty(FLUSH_BYTES // 4, dtype=torch.float32, device=dev)

    noisy = bool(cfg.get("noise"))  # configs[3]: per-wire noise rides the inverse row transform (step a7)

    def step():
        plan.clear()
        plan.raster_scatter(d, seed=cfg["fluct_seed"], fluctuate=fluct)
        if noisy:
            plan.arm_noise(None, seed=cfg["noise_seed"])
        plan.convolve()

    def timed(fn, k, sampler=None):
        """k steps; L2 flushed before each; returns the per-step device times in ms (CUDA events on the stream)."""
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(k)]
        replicas.barrier()
        torch.cuda.synchronize()
        if sampler:
            sampler.start()
        for a, b in ev:
            flush.fill_(1.0)
            a.record(stream)
            fn()
            b.record(stream)
        if sampler:
            sampler.sample()
        torch.cuda.synchronize()
        if sampler:
            sampler.stop()
        replicas.barrier()
        return [a.elapsed_time(b) for a, b in ev]

    # ---- device-resident arm -------------------------------------------------------------------------------------
    # The headline is timed with one CUDA-event pair per plane-event and nothing between the kernels.  The per-kernel
    # durations of the roofline come from a second pass of the same K steps with the library's own event pairs around
    # every stage (wcsim_set_profiling): those records sit between the kernels and cost ~20 us per step on
    # configs[1], so they are kept out of the headline and reported as ms_per_step_with_stage_events.
    for _ in range(args.warmup):
        flush.fill_(1.0)
        step()
    torch.cuda.synchronize()
    plan.reset_stats()
    launches0 = plan.launch_count()
    sampler = ClockSampler(nvml_index(local_rank))
    per_step = timed(step, args.steps, sampler)
    launches = plan.launch_count() - launches0
    local_s = sum(per_step) * 1e-3
    value, slowest_s = replicas.whole_job_throughput(n_depos * args.steps, local_s, dev)
    ms_per_step = slowest_s * 1e3 / args.steps

    # the same K steps without the convolution: what the convolve stage adds to a back-to-back plane-event (its kernels
    # are programmatic dependents of the raster and of one another, so this is less than the sum of their stand-alone times)
    def step_raster_only():
        plan.clear()
        plan.raster_scatter(d, seed=cfg["fluct_seed"], fluctuate=fluct)

    for _ in range(min(args.warmup, 3)):
        flush.fill_(1.0)
        step_raster_only()
    per_step_raster = timed(step_raster_only, args.steps)
    ms_raster_only = sum(per_step_raster) / len(per_step_raster)

    # stage durations, two ways: (1) one event pair around each CALL (raster; the whole wcsim_convolve with nothing recorded
    # between its three kernels, which stay programmatic dependents of one another): the convolve stage as it runs inside
    # the back-to-back plane-event; (2) one pair around every KERNEL: the per-kernel figures
    def staged_pass(level):
        plan.set_profiling(level)
        for _ in range(min(args.warmup, 3)):
            flush.fill_(1.0)
            step()
        torch.cuda.synchronize()
        plan.stage_times(reset=True)
        per = timed(step, args.steps)
        st = plan.stage_times(reset=True)
        plan.set_profiling(0)
        return per, st

    per_step_calls, stages_calls = staged_pass(B.WCSIM_PROFILE_CALLS)
    per_step_staged, stages = staged_pass(B.WCSIM_PROFILE_KERNELS)
    stats = plan.stats()

    # ---- end to end through the C ABI with host buffers -------------------------------------------------------------
    # Every step copies its depos host->device and its M device->host (pinned buffers) inside the timed region.  Three
    # plans on three streams are used in turn through wcsim_simulate_host_async, so the 19 MB device->host copy of
    # one plane-event runs under the next event's copies and kernels; a step's M is on the host when its plan is
    # synchronised, which happens before that plan is reused and, for the last steps, before the clock stops.
    # the five depo arrays in ONE pinned block: wcsim_simulate_host*_async then sends them in a single copy
    host_block = torch.empty(5 * n_depos, dtype=torch.float32).pin_memory()
    host = {}
    for a_, k_ in enumerate(("t0", "x0", "sigma_t", "sigma_x", "q")):
        host[k_] = host_block[a_ * n_depos:(a_ + 1) * n_depos]
        host[k_].copy_(torch.from_numpy(pl["depos"][k_]))
    n_e2e_plans = 3  # two leave the device->host engine idle part of the time (436 us); four gain nothing over three
    e2e_streams = [torch.cuda.Stream(device=dev) for _ in range(n_e2e_plans)]
    e2e_plans = [make_plan(st) for st in e2e_streams]
    host_M = [torch.empty((pl["n_wires"], pl["n_ticks"]), dtype=torch.float32).pin_memory() for _ in range(n_e2e_plans)]

    def run_e2e(k):
        for i in range(k):
            p = e2e_plans[i % n_e2e_plans]
            p.sync()  # the plane-event this plan ran n_e2e_plans steps ago is complete: its host_M may be overwritten
            p.simulate_host_async(host, host_M[i % n_e2e_plans], seed=cfg["fluct_seed"], fluctuate=fluct)
        for p in e2e_plans:
            p.sync()

    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    run_e2e(max(2, min(args.warmup, 3)))
    replicas.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    run_e2e(e2e_steps)
    torch.cuda.synchronize()
    e2e_local = time.perf_counter() - t0
    replicas.barrier()
    e2e_value, e2e_slowest = replicas.whole_job_throughput(n_depos * e2e_steps, e2e_local, dev)
    h2d, d2h = 5 * 4 * n_depos, 4 * pl["n_wires"] * pl["n_ticks"]
    # the synchronous call, one plane-event at a time (latency of the whole host round trip)
    plan.simulate_host(host, host_M[0], seed=cfg["fluct_seed"], fluctuate=fluct)  # allocates the plan's staging arrays
    t0 = time.perf_counter()
    for _ in range(min(e2e_steps, 20)):
        plan.simulate_host(host, host_M[0], seed=cfg["fluct_seed"], fluctuate=fluct)
    e2e_sync_ms = (time.perf_counter() - t0) * 1e3 / min(e2e_steps, 20)
    # extra: the same round trip returning 12-bit ADC codes (wcsim_simulate_host_adc_async, reading A23) instead of the
    # fp32 M: half the device->host bytes; every step's codes are on the host when its plan is synchronised
    host_adc = [torch.empty((pl["n_wires"], pl["n_ticks"]), dtype=torch.int16).pin_memory() for _ in range(n_e2e_plans)]

    def run_e2e_adc(k):
        for i in range(k):
            j = i % n_e2e_plans
            p = e2e_plans[j]
            p.sync()
            p.simulate_host_adc_async(host, host_adc[j], ADC_GAIN, ADC_BASELINE, 12, seed=cfg["fluct_seed"], fluctuate=fluct)
        for p in e2e_plans:
            p.sync()

    run_e2e_adc(2)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    run_e2e_adc(e2e_steps)
    torch.cuda.synchronize()
    e2e_adc_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
    for p in e2e_plans:
        p.destroy()

    # ---- several independent plane-events in flight (the paper's section 3.3 runs several processes
    # per GPU for the same reason: one event does not fill the device).  Extra figure, not the headline.
    concurrent = batched = graphed = None
    if args.streams > 1 and world == 1 and args.impact == 1:
        concurrent = concurrent_planes(args, B, cfg, pl, d, fluct, mode, dev, n_depos)
        if len(cfg["planes"]) == 1:
            # the same number of independent plane-events through ONE launch sequence of a multi-plane plan
            batched = batched_events(args, B, cfg, [pl] * args.streams, [d] * args.streams, fluct, mode, dev)
            batched["ms_per_plane_event"] = batched["ms_per_event"] / args.streams
            batched["ms_per_plane_event_cuda_graph"] = batched["ms_per_event_cuda_graph"] / args.streams
    if world == 1 and args.impact == 1:
        graphed = graph_plane_event(args, B, cfg, pl, d, fluct, mode, dev, flush)

    # configs[3] is an APA event: three planes with their own responses, noise on every one.  Extra figure: whole events,
    # the three planes of an event on three plans/streams (planes are independent)
    apa = None
    if len(cfg["planes"]) > 1 and world == 1 and args.impact == 1:
        apa = apa_events(args, B, cfg, fluct, mode, dev)

    # ---- roofline of the dominant kernel --------------------------------------------------------------------------
    peaks = load_peaks()
    direct = plan.wire_mode() == B.WCSIM_WIRES_DIRECT  # the route the library resolved (wcsim_get_wire_mode), not a copy of its rule
    sb = stage_bytes(pl, direct, args.impact)
    stage_rows = []
    for name in ("raster", "rows_forward", "cols", "rows_inverse"):
        ms, calls = stages[name]
        if calls == 0:
            continue
        avg = ms / calls
        row = {"stage": name, "ms": avg}
        if name in sb:
            gbs = sb[name] / (avg * 1e-3) / 1e9
            row.update({"bound": "hbm", "bytes": sb[name], "achieved_gbs": gbs, "frac": gbs / peaks["hbm_gbs"]})
        else:
            row.update({"bound": "alu", "depos_per_s": n_depos / (avg * 1e-3)})
        stage_rows.append(row)
    conv_sum_ms = sum(r["ms"] for r in stage_rows if r["stage"] in sb)
    conv_bytes = sum(sb.values())
    pass_model = survey_pass_model_bytes(pl)

    def hbm_fracs(ms):
        gbs = conv_bytes / (ms * 1e-3) / 1e9
        return {"ms": ms, "achieved": gbs, "frac": gbs / peaks["hbm_gbs"],
                "frac_of_survey_pass_model": pass_model / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"]}

    # Headline of the stage: ONE event pair around the whole wcsim_convolve call inside the back-to-back plane-event (the
    # raster precedes it, nothing is recorded between its three kernels); `frac` counts the bytes the kernels actually move.
    # SURVEY.md 8(d)'s pass model (all three passes by FFT, Rhat read in full: 33 MB more on configs[1], which the direct
    # wire-axis pass never reads) is the labelled secondary figure.
    c_ms, c_calls = stages_calls["convolve"]
    convolve = hbm_fracs(c_ms / max(c_calls, 1))
    # compulsory floor: S read once, Rhat read once, M written once -- no intermediate spectrum traffic
    floor_bytes = 2 * pl["n_wires"] * pl["n_ticks"] * 4 + pl["pad_w"] * (pl["pad_t"] // 2 + 1) * 8
    floor_ms = floor_bytes / (peaks["hbm_gbs"] * 1e9) * 1e3
    convolve.update({"compulsory_floor": {"bytes": floor_bytes, "ms_at_peak": floor_ms, "frac": floor_ms / convolve["ms"],
                                          "what": "read S + read Rhat + write M at the measured copy bandwidth, over the measured time"}})
    convolve.update({"bytes": conv_bytes, "survey_pass_model_bytes": pass_model,
                     "how": "one CUDA-event pair around wcsim_convolve in the back-to-back plane-event",
                     "frac_of_8TBs_nominal": convolve["achieved"] / 8000.0,
                     "kernels_timed_one_by_one": hbm_fracs(conv_sum_ms)})
    if world == 1 and ms_per_step - ms_raster_only > 0:
        # plane-event minus (clear + raster) timed alone: what the stage adds to the pipeline (two separately timed loops)
        convolve["plane_event_minus_raster"] = dict(hbm_fracs(ms_per_step - ms_raster_only),
                                                    ms_clear_and_raster_alone=ms_raster_only)
    dom = max(stage_rows, key=lambda r: r["ms"])
    if dom["stage"] == "raster" and fluct:
        # ALU bound: algorithmic fp64 work of the oracle's arithmetic, ~70 flop per drawn bin,
        # against 148 SMs x 64 fp64 FMA lanes x 2 flop x the SM clock
        bins = stats["bins_drawn"] / max(1, 4 * args.steps + 3 * min(args.warmup, 3))  # plane-events since the reset
        tflops = bins * FP64_FLOP_PER_BIN / (dom["ms"] * 1e-3) / 1e12
        peak = 148 * 64 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
        roofline = {"kernel": "raster_batch_kernel<fluct>", "bound": "alu", "achieved": tflops, "peak": peak,
                    "unit": "TFLOP/s", "frac": tflops / peak, "traffic": TRAFFIC.get("raster") if args.config == 1 else None,
                    "peak_source": "derived, not measured in this run: 148 SMs x 64 fp64 FMA/clk x 2 x %.0f MHz (DESIGN.md); a DFMA "
                                   "microbenchmark reached 56.4 of 64 per clk per SM in round 1" % peaks["sm_max_mhz"],
                    "algorithmic": {"bins_per_launch": bins, "fp64_flop_per_bin": FP64_FLOP_PER_BIN,
                                    "bins_per_s": bins / (dom["ms"] * 1e-3)}}
        # the informative roof (the kernel is issue bound, not fp64 bound): warp-instructions per drawn bin as ncu counted
        # them on this workload (smsp__inst_executed.sum / bins; profiles/r02_ncu_full.md: 35.77 M / 2,127,063) against 4 per clock per SM
        issue_peak = 148 * 4 * peaks["sm_max_mhz"] * 1e6
        issued = bins * WARP_INST_PER_BIN / (dom["ms"] * 1e-3)
        roofline["issue"] = {"warp_instructions_per_bin": WARP_INST_PER_BIN if args.config == 1 else None,
                             "achieved_warp_inst_per_s": issued if args.config == 1 else None, "peak_warp_inst_per_s": issue_peak,
                             "frac": issued / issue_peak if args.config == 1 else None,
                             "source": "instruction count from the committed ncu capture of configs[1] (a constant here, not "
                                       "re-measured in this run); peak derived: 148 SMs x 4 schedulers x %.0f MHz" % peaks["sm_max_mhz"]}
    else:
        if dom["stage"] not in sb:
            dom = max((r for r in stage_rows if r["stage"] in sb), key=lambda r: r["ms"])
        roofline = {"kernel": dom["stage"], "bound": "hbm", "achieved": dom["achieved_gbs"], "peak": peaks["hbm_gbs"],
                    "unit": "GB/s", "frac": dom["frac"], "traffic": TRAFFIC.get(dom["stage"]) if args.config == 1 else None,
                    "peak_source": peaks["source"]}
    roofline["hbm_peak"] = {"gbs": peaks["hbm_gbs"], "source": peaks["source"]}
    roofline["convolve"] = convolve
    roofline["stages"] = stage_rows

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if not fluct else "f32 (f64 fluctuation weights and sampler)", "data": "synthetic",
        "config": {"workload": cfg["name"] + (", fluctuation off" if not fluct else ", normal-approximation fluctuation" if fluct == 2
                                             else ", fluctuation on") +
                               (", noise fused (plane 0 timed)" if noisy else "") +
                               (", LARGE-PATCH VARIANT sigma x %g (not one of the five configs)" % args.sigma_scale
                                if args.sigma_scale != 1.0 else "") +
                               (", depos in SHUFFLED order (sensitivity run)" if args.shuffle else "") +
                               (", IMPACT-POSITION VARIANT: %d impact positions per wire, reading A25 (not one of the five "
                                "configs)" % args.impact if args.impact > 1 else ""),
                   "grid": [pl["n_wires"], pl["n_ticks"]], "pad": [pl["pad_w"], pl["pad_t"]],
                   "response": list(pl["response"].shape), "depos": n_depos, "scatter": args.scatter,
                   "wire_axis": "direct" if direct else "fft",
                   "parallelism": "replicas x%d" % world, "l2": "flushed between timed steps (256 MB write)"},
        "clocks": sampler.summary(),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_slowest * 1e3 / e2e_steps, "steps": e2e_steps,
                "how": "wcsim_simulate_host_async on %d plans/streams in turn, pinned host buffers" % n_e2e_plans,
                "ms_per_step_synchronous_call": e2e_sync_ms,
                "adc_variant": {"ms_per_step": e2e_adc_ms, "value": n_depos / (e2e_adc_ms * 1e-3),
                                "d2h_bytes_per_step": d2h // 2,
                                "what": "wcsim_simulate_host_adc_async: 12-bit ADC codes (int16) come back instead of fp32 M"}},
        "gpu_launches": launches,
        "build": build_identity(B),
        "roofline": roofline,
        "ms_per_step_median": statistics.median(per_step),
        "ms_per_step_min": min(per_step),
        "ms_per_step_with_call_events": sum(per_step_calls) / len(per_step_calls),
        "ms_per_step_with_kernel_events": sum(per_step_staged) / len(per_step_staged),
    }
    if concurrent:
        out["concurrent"] = concurrent
    if batched:
        out["batched"] = batched
    if graphed:
        out["cuda_graph"] = graphed
    if apa:
        out["apa_event"] = apa
    if rank == 0 and world == 1 and not args.no_cpu_baseline and args.impact == 1:
        out["cpu_baseline"] = cpu_baseline(cfg, budget_s=args.cpu_budget)
    if rank == 0 and world == 1 and not args.no_cufft:
        out["cufft_comparator"] = cufft_comparator(pl, dev, flush)
    plan.destroy()
    replicas.shutdown()
    if rank == 0:
        print(json.dumps(out))


# dram__bytes_read.sum + dram__bytes_write.sum per launch on configs[1], from the committed `ncu --set full` capture
# (profiles/r02_ncu_full.md; cold-cache replays, so reads are compulsory misses and writes mostly stay in L2)
TRAFFIC = {"raster": 5.96e6, "rows_forward": 19.29e6, "cols": 27.70e6, "rows_inverse": 26.36e6}
# warp-instructions per drawn bin of the fluctuated raster on configs[1] (ncu: smsp__inst_executed.sum / 2,127,063 bins)
WARP_INST_PER_BIN = 16.8
# algorithmic fp64 work per drawn bin of the fluctuated raster (DESIGN.md section 6 derives it from the oracle's steps)
FP64_FLOP_PER_BIN = 70.0
# the e2e ADC variant's ideal converter (reading A23): codes per unit of M, and pedestal
ADC_GAIN, ADC_BASELINE = 0.01, 900.0


def build_identity(B):
    """Which libwcsim.so was timed: its version string and a hash of the file, so that the constants typed in above from one
    ncu capture (TRAFFIC, WARP_INST_PER_BIN) can be matched against the build named in the header of profiles/r03_*.md."""
    import hashlib
    from paper_2203_02479_b200 import build as _b
    with open(_b.LIB, "rb") as f:
        digest = hashlib.sha256(f.read()).hexdigest()
    return {"version": B.wcsim_version(), "libwcsim_sha256_16": digest[:16],
            "ncu_constants_from": "profiles/r02_ncu_full.md (round-2 build; the raster kernels are unchanged since)"}


def survey_pass_model_bytes(pl):
    """read S, write+read the populated row spectra twice, read Rhat, write M."""
    nw, nt, pw, pt = pl["n_wires"], pl["n_ticks"], pl["pad_w"], pl["pad_t"]
    nk = pt // 2 + 1
    return 2 * nw * nt * 4 + 4 * nw * nk * 8 + pw * nk * 8


def concurrent_planes(args, B, cfg, pl, d, fluct, mode, dev, n_depos):
    """K plane-events of the same workload issued round-robin to `--streams` plans, each with its own stream and
    buffers (working set n x 90 MB > L2 for n >= 2, so no flush); one CUDA-event pair around all K."""
    import torch
    n = args.streams
    streams = [torch.cuda.Stream(device=dev) for _ in range(n)]
    plans = [B.Plan(pl["n_wires"], pl["n_ticks"], pl["response"], pad=(pl["pad_w"], pl["pad_t"]), nsigma=cfg["nsigma"],
                    scatter_mode=mode, stream=st) for st in streams]
    main = torch.cuda.current_stream()

    def run(k):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record(main)
        for st in streams:
            st.wait_event(a)
        for i in range(k):
            p = plans[i % n]
            p.clear()
            p.raster_scatter(d, seed=cfg["fluct_seed"], fluctuate=fluct)
            p.convolve()
        for st in streams:
            main.wait_stream(st)
        b.record(main)
        torch.cuda.synchronize()
        return a.elapsed_time(b)

    run(max(n, min(args.warmup, 3) * n))
    ms = run(args.steps)
    for p in plans:
        p.destroy()
    return {"streams": n, "steps": args.steps, "ms_per_step": ms / args.steps, "value": n_depos * args.steps / (ms * 1e-3),
            "unit": UNIT, "what": "independent plane-events in flight on %d streams (throughput, not latency)" % n}


def apa_events(args, B, cfg, fluct, mode, dev):
    """K whole events of a multi-plane config, two ways: plane p of every event on its own plan/stream (round 1's way),
    and all planes through ONE launch sequence of a multi-plane plan (wcsim_plan_create_planes: one raster launch, row
    transforms over the stacked rows, one wire pass), issued call by call and replayed from a CUDA graph."""
    import torch
    planes = cfg["planes"]
    streams = [torch.cuda.Stream(device=dev) for _ in planes]
    plans = [B.Plan(pl["n_wires"], pl["n_ticks"], pl["response"], pad=(pl["pad_w"], pl["pad_t"]), nsigma=cfg["nsigma"],
                    scatter_mode=mode, stream=st) for pl, st in zip(planes, streams)]
    depos = [{k: torch.from_numpy(v).to(dev) for k, v in pl["depos"].items()} for pl in planes]
    n_depos = sum(int(pl["depos"]["t0"].shape[0]) for pl in planes)
    main = torch.cuda.current_stream()

    def run(k):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record(main)
        for st in streams:
            st.wait_event(a)
        for _ in range(k):
            for p, d, pl in zip(plans, depos, planes):  # every plane with its own seeds (reading A26)
                p.clear()
                p.raster_scatter(d, seed=pl["fluct_seed"], fluctuate=fluct)
                if cfg.get("noise"):
                    p.arm_noise(None, seed=pl["noise_seed"])
                p.convolve()
        for st in streams:
            main.wait_stream(st)
        b.record(main)
        torch.cuda.synchronize()
        return a.elapsed_time(b)

    run(3)
    ms = run(args.steps)
    for p in plans:
        p.destroy()
    out = {"planes": len(planes), "depos_per_event": n_depos, "events": args.steps, "ms_per_event": ms / args.steps,
           "value": n_depos * args.steps / (ms * 1e-3), "unit": UNIT,
           "what": "whole events, plane p on plan/stream p (raster + fused noise + convolve per plane)"}
    out["batched"] = batched_events(args, B, cfg, planes, depos, fluct, mode, dev)
    return out


def batched_events(args, B, cfg, planes, depos, fluct, mode, dev):
    """K events, all planes of an event through one launch sequence of a multi-plane plan; call by call and as a CUDA graph."""
    import torch
    n_depos = sum(int(d["t0"].numel()) for d in depos)
    st = torch.cuda.Stream(device=dev)
    bmode = mode if mode != B.WCSIM_SCATTER_TILED else B.WCSIM_SCATTER_FIXED  # the tiled mode is per plane
    plan = B.PlanesPlan([pl["n_wires"] for pl in planes], planes[0]["n_ticks"], [pl["response"] for pl in planes],
                        pad_ticks=planes[0]["pad_t"], nsigma=cfg["nsigma"], scatter_mode=bmode, stream=st)

    # a seed per plane (reading A26); copies of one plane (--streams) get distinct seeds too
    fluct_seeds = [pl["fluct_seed"] + 0x100000 * i for i, pl in enumerate(planes)]
    noise_seeds = [pl["noise_seed"] + 0x100000 * i for i, pl in enumerate(planes)]

    def event():
        plan.clear()
        plan.raster_scatter_planes(depos, seeds=fluct_seeds, fluctuate=fluct)
        if cfg.get("noise"):
            plan.arm_noise_planes(None, seeds=noise_seeds)
        plan.convolve()

    def run(fn, k):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record(st)
        for _ in range(k):
            fn()
        b.record(st)
        torch.cuda.synchronize()
        return a.elapsed_time(b)

    run(event, 3)
    l0 = plan.launch_count()
    ms_calls = run(event, args.steps)
    launches = (plan.launch_count() - l0) / args.steps
    plan.graph_begin()
    event()
    graph = plan.graph_end()
    run(graph.launch, 3)
    ms_graph = run(graph.launch, args.steps)
    graph.destroy()
    plan.destroy()
    return {"planes": len(planes), "depos_per_event": n_depos, "events": args.steps, "kernel_launches_per_event": launches,
            "ms_per_event": ms_calls / args.steps, "value": n_depos * args.steps / (ms_calls * 1e-3),
            "ms_per_event_cuda_graph": ms_graph / args.steps, "value_cuda_graph": n_depos * args.steps / (ms_graph * 1e-3),
            "unit": UNIT, "what": "all planes of an event through one launch sequence of a multi-plane plan "
                                  "(wcsim_plan_create_planes), events back to back, no L2 flush"}


def graph_plane_event(args, B, cfg, pl, d, fluct, mode, dev, flush):
    """The headline plane-event replayed from a CUDA graph on its own stream (clear, raster, convolve recorded once):
    per-step CUDA-event pairs, L2 flushed before each step as in the headline."""
    import torch
    st = torch.cuda.Stream(device=dev)
    if mode == B.WCSIM_SCATTER_TILED:
        return None
    plan = B.Plan(pl["n_wires"], pl["n_ticks"], pl["response"], pad=(pl["pad_w"], pl["pad_t"]), nsigma=cfg["nsigma"],
                  scatter_mode=mode, stream=st)

    def event():
        plan.clear()
        plan.raster_scatter(d, seed=cfg["fluct_seed"], fluctuate=fluct)
        if cfg.get("noise"):
            plan.arm_noise(None, seed=cfg["noise_seed"])
        plan.convolve()

    event()  # first use allocates what the mode needs
    plan.sync()
    plan.graph_begin()
    event()
    graph = plan.graph_end()

    def timed(fn, k):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(k)]
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            for a, b in ev:
                flush.fill_(1.0)
                a.record(st)
                fn()
                b.record(st)
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in ev]

    timed(graph.launch, 3)
    per_graph = timed(graph.launch, args.steps)
    per_calls = timed(event, args.steps)
    graph.destroy()
    plan.destroy()
    return {"ms_per_step": sum(per_graph) / len(per_graph), "ms_per_step_median": statistics.median(per_graph),
            "ms_per_step_same_stream_call_by_call": sum(per_calls) / len(per_calls),
            "what": "the same plane-event replayed from a CUDA graph (wcsim_graph_*), L2 flushed between steps"}


def cufft_comparator(pl, dev, flush):
    """cuFFT (through torch.fft) R2C -> pointwise multiply -> C2R on the same padded sizes: comparator only."""
    import torch
    nw, nt, pw, pt = pl["n_wires"], pl["n_ticks"], pl["pad_w"], pl["pad_t"]
    S = torch.rand((nw, nt), device=dev)
    Rh = torch.fft.rfft2(torch.rand((pw, pt), device=dev))
    ms = []
    for it in range(8):
        flush.fill_(1.0)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        M = torch.fft.irfft2(torch.fft.rfft2(S, s=(pw, pt)) * Rh, s=(pw, pt))[:nw, :nt]
        b.record()
        torch.cuda.synchronize()
        if it >= 3:
            ms.append(a.elapsed_time(b))
    return {"ms": statistics.median(ms), "what": "torch.fft.rfft2 (cuFFT) * Rhat -> irfft2, crop; comparator only"}


# --------------------------------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline leg and --impl reference)
# --------------------------------------------------------------------------------------------------------------------
def oracle_step(cfg, O):
    """One plane-event of the workload through oracle/ as it stands: raster+fluctuate+scatter, FFT-route convolve."""
    pl = cfg["planes"][0]
    S, _, _ = O.raster_scatter(pl["n_wires"], pl["n_ticks"], pl["depos"], seed=cfg["fluct_seed"],
                               fluctuate=cfg["fluctuate"], nsigma=cfg["nsigma"])
    return O.convolve_fft(S, pl["response"], pl["pad_w"], pl["pad_t"])


def cpu_baseline(cfg, budget_s=15.0):
    import oracle as O
    O.lib()
    n_depos = int(cfg["planes"][0]["depos"]["t0"].shape[0])
    oracle_step(cfg, O)  # page in
    t0 = time.perf_counter()
    reps = 0
    while reps < 1 or (time.perf_counter() - t0 < budget_s and reps < 50):
        oracle_step(cfg, O)
        reps += 1
    dt = time.perf_counter() - t0
    cores = O.num_threads()
    out = {"value": n_depos * reps / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
           "ms_per_step": dt * 1e3 / reps,
           "sample": "%d whole plane-events of the same workload (all %d depos, full grid), fp64, "
                     "FFT-route convolution" % (reps, n_depos)}
    # per stage, all cores (one plane-event): raster + fluctuation + serial scatter, FFT-route convolution
    pl = cfg["planes"][0]
    t0 = time.perf_counter()
    S, _, _ = O.raster_scatter(pl["n_wires"], pl["n_ticks"], pl["depos"], seed=cfg["fluct_seed"],
                               fluctuate=cfg["fluctuate"], nsigma=cfg["nsigma"])
    t1 = time.perf_counter()
    O.convolve_fft(S, pl["response"], pl["pad_w"], pl["pad_t"])
    t2 = time.perf_counter()
    out["stages_ms"] = {"raster_scatter": (t1 - t0) * 1e3, "convolve_fft": (t2 - t1) * 1e3}
    # one thread, what the paper's CPU-ref was: one plane-event
    O.set_num_threads(1)
    t0 = time.perf_counter()
    oracle_step(cfg, O)
    dt1 = time.perf_counter() - t0
    O.set_num_threads(cores)
    out["single_thread"] = {"value": n_depos / dt1, "ms_per_step": dt1 * 1e3, "cores": 1, "sample": "1 whole plane-event"}
    return out


def run_reference(args):
    """The reference arm of this tier is the oracle (there is no reference code): timed on the host, rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2203_02479_b200 import synth
    import oracle as O
    O.lib()
    cfg = synth.config(args.config)
    pl = cfg["planes"][0]
    n_depos = int(pl["depos"]["t0"].shape[0])
    steps = max(1, min(args.steps, args.ref_max_steps))
    for _ in range(max(1, min(args.warmup, 2))):
        oracle_step(cfg, O)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle_step(cfg, O)
    dt = time.perf_counter() - t0
    value = n_depos * steps / dt
    sample = ("each step = one whole plane-event of the workload (all %d depos, full grid); %d of the %d requested "
              "steps run to stay within minutes" % (n_depos, steps, args.steps))
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3 / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"] + ", fluctuation on", "grid": [pl["n_wires"], pl["n_ticks"]],
                   "pad": [pl["pad_w"], pl["pad_t"]], "response": list(pl["response"].shape), "depos": n_depos,
                   "parallelism": "host cores (OpenMP)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index of the timed workload")
    ap.add_argument("--scatter", default="atomic", choices=["atomic", "tiled", "fixed"])
    ap.add_argument("--wires", default="auto", choices=["auto", "fft", "direct"], help="wire axis of the convolution")
    ap.add_argument("--no-fluct", action="store_true")
    ap.add_argument("--fluct", default="binomial", choices=["binomial", "normal"],
                    help="sampler of the fluctuated raster: reading A6 (headline) or the Kokkos port's normal approximation (A21)")
    ap.add_argument("--sigma-scale", type=float, default=1.0,
                    help="labelled large-patch variant of configs[1]/[2] (reading A19): widths multiplied by this factor")
    ap.add_argument("--shuffle", action="store_true",
                    help="sensitivity run (SURVEY 8d): the depos in a random order instead of generation order (tracks consecutive)")
    ap.add_argument("--impact", type=int, default=1,
                    help="labelled variant (reading A25): impact positions per wire; depos and response are re-expressed on the finer grid")
    ap.add_argument("--streams", type=int, default=3, help="plane-events in flight for the extra `concurrent` figure")
    ap.add_argument("--e2e-steps", type=int, default=200)
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle time for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cufft", action="store_true", help="skip the cuFFT comparator (8 iterations of torch.fft on the padded sizes)")
    ap.add_argument("--cufft", action="store_true", help=argparse.SUPPRESS)  # old spelling: the comparator now runs by default
    ap.add_argument("--ref-max-steps", type=int, default=20)
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3  # timing rule: at least 3 warm-up steps
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
