#!/usr/bin/env python
"""bench.py -- one "step" = one pass of the whole hot path (plan tables resident; pack, every RF and
free-precession block, the two-pass signal reduction, final state) over one synthetic workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 4] [--impl ours|reference]

Prints ONE JSON line (rank 0).  metric = Bloch spin*steps/s: N_spins x N_intervals of the discretised
sequence (what the step-by-step solver of the paper executes, SURVEY.md 8(d) "Counting") / device time.
See DESIGN.md "Measurement" for the roofline arithmetic.  The reference arm (--impl reference) times the
fp64 CPU oracle, as it stands, on the host cores; it is the only place besides cpu_baseline that touches
oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
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
# DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) from the committed ncu --set full captures
NCU_TRAFFIC = {("config4_1M_spiral", "signal"): (32.08e6, "profiles/r01_v3_signal_kernel_cfg4_ncu.txt"),
               ("config4_1M_spiral", "rf"): (48.11e6, "profiles/r01_v3_rf_kernel_cfg4_ncu.txt"),
               ("config3_brain_epi128", "signal"): (6.57e6, "profiles/r01_v4_signal_lin_kernel_cfg3_ncu.txt"),
               ("config5_mrf_fisp", "fused"): (1229.9e6, "profiles/r01_v3_seq_kernel_cfg5_ncu.txt")}


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


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
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def make_workload(name: str, rank: int):
    """Rank r simulates shard r of an (N x n_spins)-spin phantom on the SAME sequence: the phantom comes from
    the same generator with the seed moved by the rank (weak scaling: per-GPU work is fixed)."""
    from paper_2301_02702_b200 import workloads as W
    w = W.make(name)
    if rank:
        base = W.SEED0
        try:
            W.SEED0 = base + 1000 * rank
            import dataclasses
            w = dataclasses.replace(w, phantom=W.make(name).phantom)
        finally:
            W.SEED0 = base
    return w


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
                        group_size=w.group_size)
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
    w = make_workload(args.workload, 0)
    t, _, _, _ = oracle.grid(w.seq, dt_max=w.dt_max if w.velocity is not None else 0.0)
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
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": w.name, "n_spins": w.phantom.n, "n_intervals": n_int,
                      "sample_spins_per_step": take},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                            "sample": f"{take} of {w.phantom.n} spins per step, full sequence, fp64"},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def run_ours(args, rank, local_rank, world):
    import torch
    import torch.distributed as dist
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2301_02702_b200 import build as bl
    if rank == 0:
        bl.build()
    if world > 1:
        dist.barrier()
    from paper_2301_02702_b200 import bloch
    from paper_2301_02702_b200.dist import reduce_signal

    w = make_workload(args.workload, rank)
    per_spin = w.output_mode in ("per_spin", "grouped")   # no cross-rank sum: outputs stay sharded
    t_plan0 = time.perf_counter()
    plan = bloch.Plan(w.seq, path=args.path, **w.plan_kw)
    plan.upload()
    torch.cuda.synchronize()
    plan_s = time.perf_counter() - t_plan0
    info = plan.info
    n = w.phantom.n
    n_int = info["n_intervals"]
    spin_steps = float(n) * float(n_int)
    dev = bloch.phantom_to_device(w.phantom)
    vel = None if w.velocity is None else tuple(
        torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda() for a in w.velocity)
    Mxy = torch.zeros(n, 2, dtype=torch.float32, device="cuda")
    Mz = torch.zeros(n, dtype=torch.float32, device="cuda")
    coils = None if w.coils is None else torch.from_numpy(np.ascontiguousarray(w.coils)).cuda()
    shape = plan._signal_shape(n) if coils is None else (int(coils.shape[0]), info["n_adc"])
    sig = torch.empty(shape, dtype=torch.complex64, device="cuda")
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        plan.simulate(*dev, Mxy=Mxy, Mz=Mz, init_equilibrium=True, signal=sig, velocity=vel, coils=coils)
        if not per_spin:
            reduce_signal(sig)

    for _ in range(args.warmup):
        flush.zero_()
        step()
    barrier()

    # ---- device-resident timing: K steps, L2 flushed (untimed) before each, CUDA events around each step.
    # Pass 1 (no per-kernel events) gives `value`; pass 2 repeats the same K steps with the library's per-kernel
    # CUDA events on the launching stream (they cost ~4 % on the 9000-launch MRF config) for the roofline.
    kinds_ms = {k: 0.0 for k in bloch.KINDS}
    kinds_n = {k: 0 for k in bloch.KINDS}
    clocks = ClockSampler(local_rank)
    ms_pass = {}
    with clocks:
        for taps in (False, True):
            if taps and args.no_taps:
                continue
            bloch.bloch_plan_set_profiling(plan.handle, taps)
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                  for _ in range(args.steps)]
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
    value = spin_steps * world * args.steps / (ms_total * 1e-3)
    bloch.bloch_plan_set_profiling(plan.handle, False)

    # ---- end to end through the host-buffer C-ABI entry: pinned host inputs, H2D + D2H inside the timed region
    ph = w.phantom
    pinned = [torch.from_numpy(np.ascontiguousarray(getattr(ph, k), dtype=np.float32)).pin_memory()
              for k in ("x", "y", "z", "M0", "T1", "T2", "dw")]
    h_sig = torch.empty(shape, dtype=torch.complex64).pin_memory()
    h_arrs = [p.numpy() for p in pinned]
    h_sig_np = h_sig.numpy()
    e2e_steps = max(1, min(args.steps, 5))
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
            reduce_signal(torch.from_numpy(h_sig_np).cuda())
    barrier()
    e2e_s = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
    e2e_value = spin_steps * world * e2e_steps / float(e2e_s.item())
    h2d = sum(int(a.nbytes) for a in h_arrs) + (sum(int(a.nbytes) for a in h_vel) if h_vel else 0) + \
        (int(h_coils.numel()) * 8 if h_coils is not None else 0)
    d2h = int(h_sig_np.nbytes)

    if rank != 0:
        return
    peaks = load_peaks()
    sm_max = float(clocks.max_mhz or peaks.get("sm_max_mhz") or 1965.0)
    mufu_peak = SM_COUNT * 16 * sm_max * 1e6          # MUFU ops/s
    fp32_peak = SM_COUNT * 128 * sm_max * 1e6         # FP32 instr/s
    n_eval_sig = float(n) * float(info["n_adc"])      # evaluations in the signal kernels per step
    n_coils = 0 if coils is None else int(coils.shape[0])
    n_pass = max(1, (n_coils + 3) // 4)               # the coil kernel evaluates sin / cos / ex2 once per 4 coils
    rf_steps = float(n) * float(info["n_rf_steps"])
    kern = {}
    if kinds_n["signal"]:
        dur = kinds_ms["signal"] * 1e-3 / args.steps
        ach = MUFU_PER_EVAL * n_eval_sig / dur
        kern["signal"] = {"bound": "alu", "pipe": "mufu", "achieved": ach / 1e12, "peak": mufu_peak / 1e12,
                          "unit": "Tmufu-op/s", "frac": ach / mufu_peak,
                          "traffic": NCU_TRAFFIC.get((w.name, "signal"), (None, None))[0],
                          "traffic_source": NCU_TRAFFIC.get((w.name, "signal"), (None, None))[1],
                          "coils": n_coils,
                          "note": "algorithmic count = 3 MUFU (sin, cos, ex2) per (spin, ADC sample), SURVEY.md 8(d); "
                                  "the kernel issues 2 + 1/P (P = 8 adjacent samples share one ex2; 4 in shorter blocks), so frac "
                                  "can reach 3 / 2.125 = 1.41 at a saturated MUFU pipe; on Cartesian readouts (k' advances by a constant step) the "
                                  "rotation recurrence issues 5 MUFU per P samples and the loop is issue-bound instead, so frac exceeds that",
                          "launches_per_step": kinds_n["signal"] // args.steps, "ms_per_step": dur * 1e3,
                          "avg_launch_ms": kinds_ms["signal"] / kinds_n["signal"],
                          "algorithmic_ops_per_launch": MUFU_PER_EVAL * n_eval_sig * args.steps / kinds_n["signal"]}
    if kinds_n["signal"] and n_coils > 0:
        # multi-coil receive: sin / cos / ex2 are coil-independent (3 MUFU per evaluation whatever the number of
        # coils); every coil adds one complex multiply-accumulate = 4 FP32 instructions per evaluation
        dur = kinds_ms["signal"] * 1e-3 / args.steps
        fp32_ops = (FP32_PER_EVAL + 4 * n_coils) * n_eval_sig
        if fp32_ops / fp32_peak > MUFU_PER_EVAL * n_eval_sig / mufu_peak:
            kern["signal"].update({"pipe": "fp32", "achieved": fp32_ops / dur / 1e12, "peak": fp32_peak / 1e12,
                                   "unit": "Tfp32-instr/s", "frac": fp32_ops / dur / fp32_peak,
                                   "algorithmic_ops_per_launch": fp32_ops * args.steps / kinds_n["signal"],
                                   "note": f"signal_coils_kernel, {n_coils} coils: algorithmic count = 15 + 4 x n_coils FP32 "
                                           "instructions per (spin, ADC sample) (SURVEY.md 8(d) + one complex MAC per coil); "
                                           "the 3 MUFU per evaluation are shared by all coils and are the smaller term"})
    if kinds_n["rf"]:
        dur = kinds_ms["rf"] * 1e-3 / args.steps
        ach = FP32_PER_RF_STEP * rf_steps / dur
        kern["rf"] = {"bound": "alu", "pipe": "fp32", "achieved": ach / 1e12, "peak": fp32_peak / 1e12,
                      "unit": "Tfp32-instr/s", "frac": ach / fp32_peak,
                      "traffic": NCU_TRAFFIC.get((w.name, "rf"), (None, None))[0],
                      "traffic_source": NCU_TRAFFIC.get((w.name, "rf"), (None, None))[1],
                      "note": "algorithmic count = 46 FP32 instructions per spin*step (Eq 6-9 + 11 written directly), "
                              "SURVEY.md 8(d); the tier-0 loop issues 38.5 per step on plateau-gradient tiles and reads 87 register "
                              "operands, so its hardware floor is the register file's 2 operands per lane per clock "
                              "(43.5 clocks per warp step; profiles/r01_pipe_microbench.md)",
                      "launches_per_step": kinds_n["rf"] // args.steps, "ms_per_step": dur * 1e3,
                      "avg_launch_ms": kinds_ms["rf"] / kinds_n["rf"],
                      "algorithmic_ops_per_launch": FP32_PER_RF_STEP * rf_steps * args.steps / kinds_n["rf"]}
    if kinds_n["fused"]:
        # whole-sequence kernel: excitation and readout share the SM, so both algorithmic counts land on one launch;
        # the binding pipe is the one whose count / peak is larger (FP32 on every config that takes this path)
        dur = kinds_ms["fused"] * 1e-3 / args.steps
        fp32_ops = FP32_PER_RF_STEP * rf_steps + FP32_PER_EVAL * n_eval_sig
        mufu_ops = MUFU_PER_EVAL * n_eval_sig
        t_fp32, t_mufu = fp32_ops / fp32_peak, mufu_ops / mufu_peak
        pipe, ops, peak = ("fp32", fp32_ops, fp32_peak) if t_fp32 >= t_mufu else ("mufu", mufu_ops, mufu_peak)
        ach = ops / dur
        kern["fused"] = {"bound": "alu", "pipe": pipe, "achieved": ach / 1e12, "peak": peak / 1e12,
                         "unit": "Tfp32-instr/s" if pipe == "fp32" else "Tmufu-op/s", "frac": ach / peak,
                         "traffic": NCU_TRAFFIC.get((w.name, "fused"), (None, None))[0],
                         "traffic_source": NCU_TRAFFIC.get((w.name, "fused"), (None, None))[1],
                         "note": "seq_kernel (a5-a8 in one launch): algorithmic count = 46 FP32 instructions per spin*step "
                                 "+ 15 FP32 instructions per (spin, ADC sample), SURVEY.md 8(d); the MUFU count "
                                 f"(3 per evaluation) would take {t_mufu * 1e3:.1f} ms, the FP32 count {t_fp32 * 1e3:.1f} ms",
                         "launches_per_step": kinds_n["fused"] // args.steps, "ms_per_step": dur * 1e3,
                         "avg_launch_ms": kinds_ms["fused"] / kinds_n["fused"],
                         "algorithmic_ops_per_launch": ops * args.steps / kinds_n["fused"]}
    dominant = max(kern, key=lambda k: kern[k]["ms_per_step"]) if kern else None
    roofline = dict(kern[dominant], kernel=dominant,
                    peak_source=f"derived: {SM_COUNT} SMs x lanes/SM/clk x {sm_max:.0f} MHz (DESIGN.md Roofline)") \
        if dominant else None
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f32" if info["phase_mode"] == 1 else "f32+f64phase",
           "data": "synthetic",
           "config": {"workload": w.name, "n_spins_per_gpu": n, "n_intervals": n_int,
                      "n_rf_steps": info["n_rf_steps"], "n_adc": info["n_adc"], "n_blocks": info["n_blocks"],
                      "output_mode": w.output_mode, "motion": w.velocity is not None, "coils": n_coils,
                      "path": "fused" if bloch.bloch_plan_uses_fused(plan.handle, n) else "per_block", "spin_steps_per_step": spin_steps * world,
                      "l2": "512 MiB buffer written before every timed step (untimed); per-step CUDA events",
                      "plan_create_upload_s": plan_s},
           "sim_wall_time_s": ms_total / args.steps * 1e-3,
           "clocks": clocks.summary(),
           "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                   "steps": e2e_steps, "api": "bloch_simulate_host (pinned host buffers)" if h_coils is None else
                          "bloch_simulate_host_coils (pinned host buffers)"},
           "gpu_launches": bloch.bloch_plan_last_launches(plan.handle) * args.steps,
           "ms_per_step_with_kernel_events": (ms_pass.get(True, 0.0) / args.steps) or None,
           "roofline": roofline,
           "kernels": kern,
           "ms_by_kind_per_step": {k: v / args.steps for k, v in kinds_ms.items()}}
    if args.microbench:
        out["pipe_microbench"] = {"mufu_ops_per_s": bloch.bloch_microbench(0), "ffma_per_s": bloch.bloch_microbench(1),
                                  "dfma_per_s": bloch.bloch_microbench(2),
                                  "ffma_3_distinct_regs_per_s": bloch.bloch_microbench(3)}
    if not args.no_cpu_baseline:
        cb, _, _ = time_oracle(w, n_int, args.cpu_budget)
        out["cpu_baseline"] = cb
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="4", help="config name: 1, 2, 3, 3m (3 with motion), 4 (default, 1M-spin spiral), 4c (4 with 8 receive coils), 4c32 (32 coils), 5, 5b, 5c (ensemble dictionary)")
    ap.add_argument("--path", default="auto", choices=["auto", "per_block", "fused"],
                    help="execution path (bloch_plan_set_path); auto = the library's choice")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-taps", action="store_true", help="diagnostic: no per-kernel CUDA events inside the timed steps")
    ap.add_argument("--cpu-budget", type=float, default=0.0, help="spin*steps for the cpu_baseline sample (0 = auto)")
    ap.add_argument("--microbench", action="store_true", help="also run the MUFU/FFMA/DFMA pipe micro-benchmarks")
    args = ap.parse_args()
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
