#!/usr/bin/env python
"""bench.py -- one "step" = one pass of the whole hot path (plan tables resident; pack, every RF and
free-precession block, the two-pass signal reduction, final state) over one synthetic workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 4] [--impl ours|reference]
                    [--scaling weak|strong] [--extra 1,2,3,5,5b,3m,4c,5x4 | none]

Prints ONE JSON line (rank 0).  metric = Bloch spin*steps/s: N_spins x N_intervals of the discretised
sequence (what the step-by-step solver of the paper executes, SURVEY.md 8(d) "Counting") / device time.
The headline workload is config 4 (the 1M-spin spiral); the default run also times the other named configs
(BASELINE.json: "report throughput on the five synthetic workloads") and one workload per widening row (3m: motion,
4c: 8 coils block by block on tcgen05, 5x4: 4 coils inside the whole-sequence kernel) in short runs and reports them
under "workloads".  See DESIGN.md "Measurement" for the roofline arithmetic.  The reference arm (--impl reference)
times the fp64 CPU oracle, as it stands, on the host cores; it is the only place besides cpu_baseline that
touches oracle/.
"""
from __future__ import annotations

import argparse
import glob
import hashlib
import json
import os
import re
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "bloch_spin_steps_per_s"
UNIT = "spin*steps/s"
SM_COUNT = 148
# pipe peaks derived from unit counts x max SM clock: MUFU 16 lanes/SM/clk,
# FP32 128 lanes/SM/clk
MUFU_PER_EVAL = 3          # sin, cos, ex2 per (spin, evaluated point)
FP32_PER_RF_STEP = 46      # Eq 6-9 + 11 written directly, per spin*step
FP32_PER_EVAL = 15         # FP32-pipe instructions per (spin, evaluated point)
EXTRA_DEFAULT = "1,2,3,5,5b,3m,4c,5x4"   # the five named configs + motion (f1) + coils per block / in the one launch (f2)


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


# --------------------------------------------------------------------------------------------------
# committed ncu captures (profiles/*_ncu.txt): read at run time, used only when they describe the launch
# --------------------------------------------------------------------------------------------------
_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def csrc_sha256() -> str:
    """Hash of the device code (every .cuh and internal.h under csrc/): a committed capture names the hash of the sources
    it was taken from, and describes this binary only if that is still the hash of the sources."""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2301_02702_b200", "csrc")
    for name in sorted(os.listdir(d)):
        if name.endswith(".cuh") or name == "internal.h":
            h.update(name.encode())
            with open(os.path.join(d, name), "rb") as f:
                h.update(f.read())
    return h.hexdigest()


def parse_ncu_txt(path: str):
    """One `ncu --set full` summary as committed under profiles/: 'kernel: [void ]NAME(args' then
    '  metric [unit] = value' lines.  Returns {"kernel", "grid", "block", "metrics": {name: (value, unit)}}."""
    out = {"kernel": None, "grid": None, "block": None, "metrics": {}, "file": os.path.relpath(path, ROOT), "csrc": None}
    try:
        with open(path) as f:
            for line in f:
                m = re.match(r"#\s*csrc_sha256:\s*([0-9a-f]{64})", line)
                if m:
                    out["csrc"] = m.group(1)
                    continue
                m = re.match(r"\s*kernel:\s*(?:void\s+)?([^()]+)\(", line)
                if m and out["kernel"] is None:
                    out["kernel"] = m.group(1).replace("bloch::", "").replace(" ", "")
                    continue
                m = re.match(r"\s*([A-Za-z0-9_.]+)\s*\[([^\]]*)\]\s*=\s*([-+0-9.eE]+)\s*$", line)
                if m:
                    out["metrics"][m.group(1)] = (float(m.group(3)), m.group(2))
    except OSError:
        return None
    g, b = out["metrics"].get("launch__grid_size"), out["metrics"].get("launch__block_size")
    out["grid"], out["block"] = (int(g[0]) if g else None), (int(b[0]) if b else None)
    return out


def find_capture(kernel: dict):
    """The newest committed capture that describes the launch just timed: same kernel name, grid and block size
    (bloch_plan_last_kernel) AND taken from the device sources as they stand (the `# csrc_sha256:` line of the capture
    equals the hash of csrc/*.cuh now).  Anything else -- another kernel, other template arguments, another launch
    shape, sources edited since the capture, a capture without a hash -- says nothing about this binary: None."""
    if not kernel or not kernel.get("name"):
        return None
    want = kernel["name"].replace(" ", "")
    now = csrc_sha256()
    best = None
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_ncu.txt"))):
        cap = parse_ncu_txt(path)
        if cap and cap["kernel"] == want and cap["grid"] == kernel["grid"] and cap["block"] == kernel["block"] \
                and cap["csrc"] == now:
            best = cap       # sorted by name: rNN_vM -> the latest round / version wins
    return best


def capture_fields(kernel: dict, pipe: str):
    """traffic (DRAM bytes per launch), pipe_util and issue_util (fractions, <= 1) from the matching capture."""
    cap = find_capture(kernel)
    if cap is None:
        return {"traffic": None, "traffic_source": None, "pipe_util": None, "issue_util": None,
                "capture_note": f"no committed profiles/*_ncu.txt capture of {kernel.get('name')} grid {kernel.get('grid')} "
                                f"block {kernel.get('block')} was taken from the device sources as they stand "
                                f"(csrc_sha256 {csrc_sha256()[:12]}...)"}
    m = cap["metrics"]

    def nbytes(key):
        v = m.get(key)
        return v[0] * _SCALE.get(v[1], 1.0) if v else 0.0

    def pct(key):
        v = m.get(key)
        return v[0] / 100.0 if v else None
    pipe_key = {"mufu": "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
                "fp32": "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
                "tf32": "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active"}[pipe]
    have = "dram__bytes_read.sum" in m
    return {"traffic": nbytes("dram__bytes_read.sum") + nbytes("dram__bytes_write.sum") if have else None,
            "traffic_source": cap["file"], "pipe_util": pct(pipe_key),
            "issue_util": pct("smsp__issue_active.avg.pct_of_peak_sustained_active"),
            "capture_kernel": {"name": cap["kernel"], "grid": cap["grid"], "block": cap["block"]}}


class ClockSampler:
    """Samples SM clock and throttle reasons with NVML every 100 ms while running (timed region only)."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        if self._nv is not None:
            self._stop.clear()
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
            self._thr = None

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def make_workload(name: str, rank: int, world: int, scaling: str):
    """weak (default): rank r simulates shard r of a (world x n_spins)-spin phantom on the SAME sequence; the
    phantom comes from the same generator with the seed moved by the rank (per-GPU work is fixed).
    strong: every rank builds the SAME named workload and keeps the contiguous spin range dist.shard_bounds gives it
    (total work is fixed)."""
    from paper_2301_02702_b200 import workloads as W
    import dataclasses
    w = W.make(name)
    if scaling == "strong":
        from paper_2301_02702_b200.dist import shard_bounds
        lo, hi = shard_bounds(w.phantom.n, rank, world)
        idx = np.arange(lo, hi)
        vel = None if w.velocity is None else tuple(np.ascontiguousarray(a[idx]) for a in w.velocity)
        coils = None if w.coils is None else np.ascontiguousarray(w.coils[:, idx])
        return dataclasses.replace(w, phantom=w.phantom.subset(idx), velocity=vel, coils=coils), w
    if rank:
        base = W.SEED0
        try:
            W.SEED0 = base + 1000 * rank
            w = dataclasses.replace(w, phantom=W.make(name).phantom)
        finally:
            W.SEED0 = base
    return w, w


def oracle_sample(w, budget_spin_steps: float, n_intervals: int):
    """A bounded sample of the workload for the CPU oracle: every m-th spin, the full sequence."""
    n = w.phantom.n
    take = int(max(1, min(n, budget_spin_steps // max(1, n_intervals))))
    if w.group_size > 1:   # whole groups
        g = max(1, take // w.group_size)
        first = np.linspace(0, n // w.group_size - 1, g).astype(np.int64) * w.group_size
        idx = (first[:, None] + np.arange(w.group_size)[None, :]).ravel()
        take = int(idx.size)
    else:
        idx = np.linspace(0, n - 1, take).astype(np.int64)
    vel = None if w.velocity is None else tuple(np.ascontiguousarray(a[idx]) for a in w.velocity)
    coils = None if w.coils is None else np.ascontiguousarray(w.coils[:, idx]).astype(np.complex128)
    return w.phantom.subset(idx), take, vel, coils


def time_oracle(w, n_intervals: int, budget_spin_steps: float):
    import oracle
    oracle.build()
    cores = os.cpu_count() or 1
    ph, take, vel, coils = oracle_sample(w, budget_spin_steps, n_intervals)
    t0 = time.perf_counter()
    if coils is None:
        oracle.simulate(ph, w.seq, output_mode=w.output_mode, n_threads=cores, velocity=vel, dt_max=w.dt_max,
                        group_size=w.group_size, waveform=w.waveform)
    else:
        # the oracle's coil path holds the per-spin signals [spins, n_adc] in memory: feed it batches of spins
        # (spins are independent, the coil signals add) so that the batch stays below ~1 GB
        n_adc = int(np.asarray(w.seq.adc_t).size)
        step = max(1, int(1e9 // (16 * max(1, n_adc))))
        for lo in range(0, ph.n, step):
            idx = np.arange(lo, min(ph.n, lo + step))
            oracle.simulate(ph.subset(idx), w.seq, n_threads=cores, coils=coils[:, idx])
    dt = time.perf_counter() - t0
    return {"value": take * n_intervals / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{take} of {w.phantom.n} spins (evenly spaced), full sequence ({n_intervals} intervals), "
                      f"fp64, OpenMP over spins, {dt:.2f} s"}, dt, take


def run_reference(args, rank, world):
    """--impl reference: the fp64 CPU oracle, as it stands, on the host cores; rank 0 only."""
    if rank != 0:
        return
    import oracle
    w, _ = make_workload(args.workload, 0, 1, "weak")
    t, _, _, _ = oracle.grid(w.seq, dt_max=w.dt_max if w.velocity is not None else 0.0, waveform=w.waveform)
    n_int = len(t) - 1
    cores = os.cpu_count() or 1
    # size a step at ~3 s of CPU work from a short probe
    probe, dtp, take_p = time_oracle(w, n_int, 2e7)
    per_step = max(2e7, probe["value"] * 3.0)
    times = []
    take = 0
    for i in range(args.warmup + args.steps):
        res, dt, take = time_oracle(w, n_int, per_step)
        if i >= args.warmup:
            times.append(dt)
    total = float(np.sum(times))
    value = take * n_int * len(times) / total
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times),
           "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": w.name, "n_spins": w.phantom.n, "n_intervals": n_int,
                      "sample_spins_per_step": take},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                            "sample": f"{take} of {w.phantom.n} spins per step, full sequence, fp64"},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def kernel_rooflines(bloch, plan, w, n, info, kinds_ms, kinds_n, steps, sm_max, n_coils):
    """Per kernel kind: achieved = ALGORITHMIC ops per launch (SURVEY.md 8(d) per-unit figure x units) / measured
    launch duration; frac = achieved / pipe peak.  Because the kernels execute FEWER operations than the algorithmic
    count (one ex2 shared by 8 samples, rotation recurrences), frac can exceed 1; pipe_util / issue_util from the
    matching committed ncu capture are the "how busy is the pipe" numbers and never do."""
    mufu_peak = SM_COUNT * 16 * sm_max * 1e6          # MUFU ops/s
    fp32_peak = SM_COUNT * 128 * sm_max * 1e6         # FP32 instr/s
    n_eval_sig = float(n) * float(info["n_adc"])      # evaluations in the signal kernels per step
    rf_steps = float(n) * float(info["n_rf_steps"])
    kern = {}

    def entry(kind, pipe, ops, note):
        dur = kinds_ms[kind] * 1e-3 / steps
        peak = mufu_peak if pipe == "mufu" else fp32_peak
        k = bloch.bloch_plan_last_kernel(plan.handle, kind)
        e = {"bound": "alu", "pipe": pipe, "achieved": ops / dur / 1e12, "peak": peak / 1e12,
             "unit": "Tmufu-op/s" if pipe == "mufu" else "Tfp32-instr/s", "frac": ops / dur / peak,
             "frac_definition": "algorithmic ops (SURVEY.md 8(d)) / measured time / pipe peak; the kernel may execute "
                                "fewer ops than the algorithmic count, see pipe_util for the pipe's busy fraction",
             "kernel": k, "note": note, "launches_per_step": kinds_n[kind] // steps, "ms_per_step": dur * 1e3,
             "avg_launch_ms": kinds_ms[kind] / kinds_n[kind],
             "algorithmic_ops_per_launch": ops * steps / kinds_n[kind]}
        e.update(capture_fields(k, pipe))
        return e

    if kinds_n["signal"]:
        kern["signal"] = entry("signal", "mufu", MUFU_PER_EVAL * n_eval_sig,
                               "algorithmic count = 3 MUFU (sin, cos, ex2) per (spin, ADC sample); the per-sample kernel "
                               "issues 2 + 1/P (P adjacent samples share one ex2), the Cartesian recurrence kernels 5 per "
                               "P samples (issue-bound, not MUFU-bound)")
        kern["signal"]["coils"] = n_coils
        k_sig = bloch.bloch_plan_last_kernel(plan.handle, "signal")
        if n_coils > 0 and k_sig["name"].startswith("signal_coils_h_kernel"):
            # tcgen05 kernel with FP16 operands (two pieces per value, FP32 accumulation): the receive sum is a dense
            # contraction [samples x spins] x [spins x coils], complex: algorithmic 8 real flops per (spin, ADC sample,
            # coil); the kernel executes 3x that.  Peak for FP16 = the measured dense bf16 peak (same rate).
            dur = kinds_ms["signal"] * 1e-3 / steps
            flops = 8.0 * n_coils * n_eval_sig
            peaks = load_peaks()
            h_peak = float(peaks.get("bf16_tflops") or 2250.0 * 0.75) * 1e12
            e = kern["signal"]
            e.update({"bound": "tensor", "pipe": "f16", "achieved": flops / dur / 1e12, "peak": h_peak / 1e12,
                      "unit": "TFLOP/s", "frac": flops / dur / h_peak,
                      "algorithmic_ops_per_launch": flops * steps / kinds_n["signal"],
                      "peak_source": "MEASURED_PEAKS.json bf16_tflops (FP16 runs at the bf16 rate)" if peaks.get("bf16_tflops")
                                     else "fallback: 0.75 x 2250 nominal bf16 TFLOP/s",
                      "note": f"{n_coils} coils on tcgen05 (kind::f16, A operand generated into tensor memory, operands split "
                              "into two FP16 pieces scaled from measured maxima): algorithmic 8 flops per (spin, ADC sample, "
                              "coil); 2 MMAs of M128 x N x K16 per 8 spins.  The kernel is bound by GENERATING the A operand "
                              "(sin / cos / ex2 + the split: ~27 instructions per (spin, sample), issue slots 70 %), not by the "
                              "tensor pipe: see issue_util"})
            e.update(capture_fields(k_sig, "tf32"))
        elif n_coils > 0 and k_sig["name"].startswith("signal_coils_tc_kernel"):
            # tcgen05 kernel: the receive sum is a dense contraction [samples x spins] x [spins x coils], complex:
            # algorithmic 8 real flops per (spin, ADC sample, coil); the kernel executes 3x that (3xTF32).  Peak for
            # TF32 = the measured dense bf16 peak x the nominal 1/2 ratio (B200_PROFILING.md).
            dur = kinds_ms["signal"] * 1e-3 / steps
            flops = 8.0 * n_coils * n_eval_sig
            peaks = load_peaks()
            tf32_peak = 0.5 * float(peaks.get("bf16_tflops") or 2250.0 * 0.75) * 1e12
            e = kern["signal"]
            e.update({"bound": "tensor", "pipe": "tf32", "achieved": flops / dur / 1e12, "peak": tf32_peak / 1e12,
                      "unit": "TFLOP/s", "frac": flops / dur / tf32_peak,
                      "algorithmic_ops_per_launch": flops * steps / kinds_n["signal"],
                      "peak_source": "MEASURED_PEAKS.json bf16_tflops x 0.5 (nominal TF32 : BF16 ratio)" if peaks.get("bf16_tflops")
                                     else "fallback: 0.75 x 2250 nominal bf16 TFLOP/s x 0.5",
                      "note": f"{n_coils} coils on tcgen05 (kind::tf32, A operand generated into tensor memory): algorithmic "
                              "8 flops per (spin, ADC sample, coil); the instruction count (4 MMAs of M128 x N x K8 per 8 spins, "
                              "~74 clocks each whatever N) bounds the kernel, not the tensor pipe's flop rate"})
            e.update(capture_fields(k_sig, "tf32"))
        elif n_coils > 0:
            # multi-coil receive: sin / cos / ex2 are coil-independent; every coil adds one complex MAC = 4 FP32
            fp32_ops = (FP32_PER_EVAL + 4 * n_coils) * n_eval_sig
            if fp32_ops / fp32_peak > MUFU_PER_EVAL * n_eval_sig / mufu_peak:
                kern["signal"] = entry("signal", "fp32", fp32_ops,
                                       f"{n_coils} coils: algorithmic count = 15 + 4 x n_coils FP32 instructions per "
                                       "(spin, ADC sample); the 3 MUFU per evaluation are shared by all coils")
                kern["signal"]["coils"] = n_coils
    if kinds_n["rf"]:
        kern["rf"] = entry("rf", "fp32", FP32_PER_RF_STEP * rf_steps,
                           "algorithmic count = 46 FP32 instructions per spin*step (Eq 6-9 + 11 written directly); the "
                           "small-angle loop (q <= 2^-14: every pulse of the configs) issues 31 FP + ~4-6 other per step (rf_const_kernel: "
                           "step records as kernel parameters, uniform operands), so frac can pass 1")
    if kinds_n["fused"]:
        # whole-sequence kernel: excitation and readout share the SM, so both algorithmic counts land on one launch;
        # the binding pipe is the one whose count / peak is larger (FP32 on every config that takes this path)
        fp32_ops = FP32_PER_RF_STEP * rf_steps + (FP32_PER_EVAL + 4 * n_coils) * n_eval_sig   # + one complex MAC per coil
        mufu_ops = MUFU_PER_EVAL * n_eval_sig
        t_fp32, t_mufu = fp32_ops / fp32_peak, mufu_ops / mufu_peak
        pipe, ops = ("fp32", fp32_ops) if t_fp32 >= t_mufu else ("mufu", mufu_ops)
        kern["fused"] = entry("fused", pipe, ops,
                              "seq_kernel (a5-a8 in one launch): algorithmic count = 46 FP32 per spin*step + 15 FP32 per "
                              f"(spin, ADC sample){' + 4 per coil (' + str(n_coils) + ' coils)' if n_coils else ''}; the MUFU count (3 per evaluation) would take {t_mufu * 1e3:.1f} ms, "
                              f"the FP32 count {t_fp32 * 1e3:.1f} ms")
    return kern


def measure(bloch, torch, dist, w, w_whole, args, steps, warmup, rank, local_rank, world, flush, clocks,
            with_e2e=True):
    """Times `steps` passes of the hot path over workload `w` (this rank's share) and returns the result dict."""
    from paper_2301_02702_b200.dist import reduce_signal
    per_spin = w.output_mode in ("per_spin", "grouped")   # no cross-rank sum: outputs stay sharded
    t_plan0 = time.perf_counter()
    plan = bloch.Plan(w.seq, path=args.path, options=args.options, **w.plan_kw)
    plan.upload()
    torch.cuda.synchronize()
    plan_s = time.perf_counter() - t_plan0
    info = plan.info
    n = w.phantom.n
    n_int = info["n_intervals"]
    n_total = w_whole.phantom.n if args.scaling == "strong" else n * world
    spin_steps_job = float(n_total) * float(n_int)
    dev = bloch.phantom_to_device(w.phantom)
    vel = None if w.velocity is None else tuple(
        torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda() for a in w.velocity)
    Mxy = torch.zeros(n, 2, dtype=torch.float32, device="cuda")
    Mz = torch.zeros(n, dtype=torch.float32, device="cuda")
    coils = None if w.coils is None else torch.from_numpy(np.ascontiguousarray(w.coils)).cuda()
    shape = plan._signal_shape(n) if coils is None else (int(coils.shape[0]), info["n_adc"])
    sig = torch.empty(shape, dtype=torch.complex64, device="cuda")
    strong = args.scaling == "strong"

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        plan.simulate(*dev, Mxy=Mxy, Mz=Mz, init_equilibrium=True, signal=sig, velocity=vel, coils=coils)
        if not per_spin:
            # the ONE collective of the path; strong scaling adds the shards in rank order, so the
            # result does not depend on the collective's algorithm
            reduce_signal(sig, deterministic=strong)

    for _ in range(warmup):
        flush.zero_()
        step()
    barrier()
    plan.status()   # raises if pack_kernel found an invalid phantom or one outside the plan's phase range

    # ---- device-resident timing: K steps, L2 flushed (untimed) before each, CUDA events around each step.
    # Pass 1 (no per-kernel events) gives `value`; pass 2 repeats the same K steps with the library's per-kernel
    # CUDA events on the launching stream (they cost ~4 % on the 9000-launch MRF config) for the roofline.
    kinds_ms = {k: 0.0 for k in bloch.KINDS}
    kinds_n = {k: 0 for k in bloch.KINDS}
    ms_pass = {}
    with clocks:
        for taps in (False, True):
            if taps and args.no_taps:
                continue
            bloch.bloch_plan_set_profiling(plan.handle, taps)
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                  for _ in range(steps)]
            barrier()
            for a, b in ev:
                flush.zero_()
                a.record()
                step()
                b.record()
                b.synchronize()
                if taps:
                    tm = bloch.bloch_plan_last_timing(plan.handle)
                    for k in bloch.KINDS:
                        kinds_ms[k] += tm["ms"][k]
                        kinds_n[k] += tm["launches"][k]
            barrier()
            ms_pass[taps] = sum(a.elapsed_time(b) for a, b in ev)
    t = torch.tensor([ms_pass[False]], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total = float(t.item())
    value = spin_steps_job * steps / (ms_total * 1e-3)
    bloch.bloch_plan_set_profiling(plan.handle, False)
    launches = bloch.bloch_plan_last_launches(plan.handle)
    fused = bloch.bloch_plan_uses_fused(plan.handle, n)

    # ---- strong scaling: the reduced signal of the sharded run must be the 1-GPU signal of the whole workload
    shard_check = None
    if strong and not per_spin and rank == 0:
        plan1 = bloch.Plan(w_whole.seq, path=args.path, options=args.options, **w_whole.plan_kw)
        d1 = bloch.phantom_to_device(w_whole.phantom)
        v1 = None if w_whole.velocity is None else tuple(
            torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda() for a in w_whole.velocity)
        c1 = None if w_whole.coils is None else torch.from_numpy(np.ascontiguousarray(w_whole.coils)).cuda()
        ref = plan1.simulate(*d1, velocity=v1, coils=c1)
        torch.cuda.synchronize()
        scale = float(ref.abs().max())
        err = float((sig - ref).abs().max()) / scale
        shard_check = {"max_err_vs_1gpu": err, "tol": 5e-6, "ok": bool(err <= 5e-6)}
        plan1.close()
        del d1, ref
        assert err <= 5e-6, f"sharded + reduced signal differs from the 1-GPU signal: {err:.3e}"

    # ---- end to end through the host-buffer C-ABI entry: pinned host inputs, H2D + D2H inside the timed region
    e2e = None
    if with_e2e:
        ph = w.phantom
        pinned = [torch.from_numpy(np.ascontiguousarray(getattr(ph, k), dtype=np.float32)).pin_memory()
                  for k in ("x", "y", "z", "M0", "T1", "T2", "dw")]
        h_sig = torch.empty(shape, dtype=torch.complex64).pin_memory()
        h_arrs = [p.numpy() for p in pinned]
        h_sig_np = h_sig.numpy()
        e2e_steps = max(1, min(steps, 5))
        h_vel = None
        if w.velocity is not None:
            pinned_v = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory() for a in w.velocity]
            h_vel = [p.numpy() for p in pinned_v]
        h_coils = None if w.coils is None else torch.from_numpy(np.ascontiguousarray(w.coils)).pin_memory()
        h_coils_np = None if h_coils is None else h_coils.numpy()

        def e2e_step():   # synchronous: returns after the D2H copy
            plan.simulate_host(*h_arrs, signal=h_sig_np, velocity=h_vel, coils=h_coils_np)

        e2e_step()   # warm-up (allocates the scratch)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
            if not per_spin and world > 1:
                reduce_signal(torch.from_numpy(h_sig_np).cuda(), deterministic=strong)
        barrier()
        e2e_s = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
        h2d = sum(int(a.nbytes) for a in h_arrs) + (sum(int(a.nbytes) for a in h_vel) if h_vel else 0) + \
            (int(h_coils.numel()) * 8 if h_coils is not None else 0)
        e2e = {"value": spin_steps_job * e2e_steps / float(e2e_s.item()), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": int(h_sig_np.nbytes), "steps": e2e_steps,
               "api": "bloch_simulate_host (pinned host buffers)" if h_coils is None else
                      "bloch_simulate_host_coils (pinned host buffers)"}

    n_coils = 0 if coils is None else int(coils.shape[0])
    sm_max = float(clocks.max_mhz or load_peaks().get("sm_max_mhz") or 1965.0)
    kern = kernel_rooflines(bloch, plan, w, n, info, kinds_ms, kinds_n, steps, sm_max, n_coils) if ms_pass.get(True) else {}
    # what the GPU evaluates (closed-form precession at ADC samples and block ends only; RF stepped): per second
    evaluated = (float(n_total) * (info["n_rf_steps"] + info["n_eval_points"])) * steps / (ms_total * 1e-3)
    res = {"workload": w.name, "value": value, "ms_per_step": ms_total / steps, "steps": steps, "warmup": warmup,
           "n_spins_per_gpu": n, "n_spins_total": n_total, "n_intervals": n_int, "n_rf_steps": info["n_rf_steps"],
           "n_adc": info["n_adc"], "n_blocks": info["n_blocks"], "output_mode": w.output_mode,
           "motion": w.velocity is not None, "coils": n_coils,
           "dtype": "f32" if info["phase_mode"] == 1 else "f32+f64phase",
           "path": "fused" if fused else "per_block", "spin_steps_per_step": spin_steps_job,
           "evaluated_units_per_s": evaluated, "plan_create_upload_s": plan_s, "e2e": e2e,
           "gpu_launches": launches * steps, "launches_per_step": launches,
           "ms_per_step_with_kernel_events": (ms_pass.get(True, 0.0) / steps) or None,
           "kernels": kern, "ms_by_kind_per_step": {k: v / steps for k, v in kinds_ms.items()},
           "shard_check": shard_check}
    plan.close()
    del dev, sig, Mxy, Mz
    torch.cuda.empty_cache()
    return res


def run_ours(args, rank, local_rank, world):
    import torch
    import torch.distributed as dist
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local_rank)
    if world > 1:
        # communicator lines ("NCCL INFO ...") are the evidence that NCCL carried the one collective of the path; the
        # JSON result stays ONE line of its own on rank 0's stdout
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2301_02702_b200 import build as bl
    if rank == 0:
        bl.build()
    if world > 1:
        dist.barrier()
    from paper_2301_02702_b200 import bloch

    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    clocks = ClockSampler(local_rank)
    w, w_whole = make_workload(args.workload, rank, world, args.scaling)
    head = measure(bloch, torch, dist, w, w_whole, args, args.steps, args.warmup, rank, local_rank, world, flush, clocks)

    # ---- the other named configs, short runs (BASELINE.json: "report throughput on the five synthetic workloads");
    # single GPU only: under torchrun the scaling arm times the headline workload alone
    extra = {}
    names = [s for s in args.extra.split(",") if s and s != "none"] if world == 1 else []
    for name in names:
        if name == args.workload:
            continue
        t0 = time.perf_counter()
        wx, wx_whole = make_workload(name, 0, 1, "weak")
        r = measure(bloch, torch, dist, wx, wx_whole, args, args.extra_steps, max(3, args.warmup), 0, local_rank, 1, flush,
                    clocks)
        r["bench_wall_s"] = time.perf_counter() - t0
        r["kernels"] = {k: {f: v[f] for f in ("pipe", "frac", "pipe_util", "issue_util", "ms_per_step", "avg_launch_ms",
                                              "launches_per_step", "kernel", "traffic", "traffic_source")}
                        for k, v in r["kernels"].items()}
        extra[name] = r

    if rank != 0:
        return
    kern = head["kernels"]
    sm_max = float(clocks.max_mhz or load_peaks().get("sm_max_mhz") or 1965.0)
    dominant = max(kern, key=lambda k: kern[k]["ms_per_step"]) if kern else None
    roofline = dict(kern[dominant], kernel_kind=dominant,
                    peak_source=f"derived: {SM_COUNT} SMs x lanes/SM/clk x {sm_max:.0f} MHz (DESIGN.md Roofline), "
                                "confirmed by bloch_microbench (profiles/r01_pipe_microbench.md); MEASURED_PEAKS.json "
                                "holds only HBM and bf16 peaks, which do not bound this path") if dominant else None
    out = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True,
           "scaling": args.scaling, "vs_baseline": None, "dtype": head["dtype"], "data": "synthetic",
           "value_definition": "step-equivalent throughput: N_spins x N_intervals of the discretised sequence (what the "
                               "paper's step-by-step solver executes) / device time; the GPU path evaluates free "
                               "precession in closed form at ADC samples and block ends only -- evaluated_units_per_s "
                               "counts (spin, RF step) + (spin, evaluated point) actually computed",
           "evaluated_units_per_s": head["evaluated_units_per_s"],
           "config": {"workload": head["workload"], "n_spins_per_gpu": head["n_spins_per_gpu"],
                      "n_spins_total": head["n_spins_total"], "n_intervals": head["n_intervals"],
                      "n_rf_steps": head["n_rf_steps"], "n_adc": head["n_adc"], "n_blocks": head["n_blocks"],
                      "output_mode": head["output_mode"], "motion": head["motion"], "coils": head["coils"],
                      "path": head["path"], "spin_steps_per_step": head["spin_steps_per_step"],
                      "sharding": ("strong: contiguous spin shards of the named workload (dist.shard_bounds) + rank-ordered "
                                   "sum of the per-rank signals" if args.scaling == "strong" else
                                   "weak: every rank simulates its own seed-shifted phantom of the named size"),
                      "l2": "512 MiB buffer written before every timed step (untimed); per-step CUDA events",
                      "plan_options": args.options, "plan_create_upload_s": head["plan_create_upload_s"]},
           "sim_wall_time_s": head["ms_per_step"] * 1e-3,
           "clocks": clocks.summary(),
           "e2e": head["e2e"],
           "gpu_launches": head["gpu_launches"],
           "ms_per_step_with_kernel_events": head["ms_per_step_with_kernel_events"],
           "roofline": roofline,
           "kernels": kern,
           "ms_by_kind_per_step": head["ms_by_kind_per_step"],
           "shard_check": head["shard_check"],
           "workloads": extra}
    if args.microbench:
        out["pipe_microbench"] = {"mufu_ops_per_s": bloch.bloch_microbench(0), "ffma_per_s": bloch.bloch_microbench(1),
                                  "dfma_per_s": bloch.bloch_microbench(2),
                                  "ffma_3_distinct_regs_per_s": bloch.bloch_microbench(3)}
    if not args.no_cpu_baseline:
        cb, _, _ = time_oracle(w_whole, head["n_intervals"], args.cpu_budget)
        out["cpu_baseline"] = cb
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="4", help="config name: 1, 2, 3, 3m (3 with motion), 3w (3 with periodic non-rigid motion), 4 (default, 1M-spin spiral), 4c (4 with 8 receive coils), 4c32 (32 coils), 5, 5b, 5c (ensemble dictionary), 5x8 (5 with 8 receive coils)")
    ap.add_argument("--path", default="auto", choices=["auto", "per_block", "fused"],
                    help="execution path (bloch_plan_set_path); auto = the library's choice")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="multi-GPU: weak = each rank its own phantom of the named size; strong = contiguous spin shards "
                         "of the ONE named workload, signals added in rank order, checked against the 1-GPU signal")
    ap.add_argument("--extra", default=EXTRA_DEFAULT,
                    help="other configs timed in short runs and reported under 'workloads' (comma list, or 'none')")
    ap.add_argument("--extra-steps", type=int, default=3)
    ap.add_argument("--option", action="append", default=[], metavar="NAME=VALUE",
                    help="diagnostic: a kernel-selection option of the plan (bloch_plan_set_option), e.g. rf_spins=2")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-taps", action="store_true", help="diagnostic: no per-kernel CUDA events inside the timed steps")
    ap.add_argument("--cpu-budget", type=float, default=0.0, help="spin*steps for the cpu_baseline sample (0 = auto)")
    ap.add_argument("--microbench", action="store_true", help="also run the MUFU/FFMA/DFMA pipe micro-benchmarks")
    args = ap.parse_args()
    args.options = {k: int(v) for k, v in (o.split("=", 1) for o in args.option)}
    from paper_2301_02702_b200.dist import env_world
    rank, local_rank, world = env_world()
    if args.cpu_budget <= 0:
        args.cpu_budget = 5e8 * max(1, (os.cpu_count() or 1))   # ~12 s at ~4e7 spin*steps/s per core (B200 host)
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    run_ours(args, rank, local_rank, world)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
