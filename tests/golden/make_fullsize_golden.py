#!/usr/bin/env python
"""Writes the full-size expected values of configs 4, 5 and 5b: the WHOLE fp64 oracle, every spin, every interval.

    python tests/golden/make_fullsize_golden.py [4] [5] [5b]        (default: all three)

Imports only ``oracle`` (the step-by-step CPU integrator) and the seeded input generators
(``paper_2301_02702_b200.workloads``, which holds none of the method's arithmetic); nothing here touches the CUDA
path.  SURVEY.md 8(d) / BASELINE.md section 2: "full-size parity is still computed once per config and cached by
input hash" -- the cache is the ``fullsize_config*.npz`` files next to this script, keyed by ``input_sha256`` (a
hash of every phantom and sequence array), which ``tests/test_gpu_fullsize_golden.py`` recomputes before it
compares the full-size GPU output element by element (Fig 3: the signal per ADC sample summed over all
spins; :244 normalisation by the reference maximum).

What is stored (fp64 results rounded to fp32 for storage: 6e-8 relative, three orders below the 1e-4 / 1e-5 bar):
  config 4   signal complex128 [65,536]; final (Mxy, Mz) of every 8th spin
  config 5   signal complex64 [1,024,000]; final (Mxy, Mz) of every spin
  config 5b  dictionary rows complex64 [100,000 entries][every 25th TR: 24, 49, ..., 999]; final (Mxy, Mz) of every entry
Cost: 1.6e11 / 2.0e11 / 2.0e11 spin*steps, i.e. about 8 / 10 / 10 minutes on 8 cores.
"""
from __future__ import annotations

import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

STATE_STRIDE = {"4": 8, "5": 1, "5b": 1}
TR_STRIDE_5B = 25


def input_sha256(w) -> str:
    """Hash of every input array of a workload (phantom SoA arrays, gradient vertices, RF samples, ADC times)."""
    h = hashlib.sha256()
    ph, s = w.phantom, w.seq
    arrs = [ph.x, ph.y, ph.z, ph.M0, ph.T1, ph.T2, ph.dw, *s.g_t, *s.g_v, s.rf_t, s.rf_dt, s.rf_re, s.rf_im, s.adc_t,
            np.array([s.t_end, s.dt_rf_max])]
    for a in arrs:
        a = np.ascontiguousarray(a, dtype=np.float64)
        h.update(str(a.shape).encode())
        h.update(a.tobytes())
    return h.hexdigest()


def golden_path(name: str) -> str:
    return os.path.join(HERE, f"fullsize_config{name}.npz")


def columns_5b(n_adc: int) -> np.ndarray:
    return np.arange(TR_STRIDE_5B - 1, n_adc, TR_STRIDE_5B, dtype=np.int64)


def make(name: str) -> None:
    import oracle
    from paper_2301_02702_b200 import workloads as W
    oracle.build()
    w = W.make(name)
    cores = os.cpu_count() or 1
    t0 = time.perf_counter()
    sig, mxy, mz = oracle.simulate(w.phantom, w.seq, output_mode=w.output_mode, return_state=True, n_threads=cores)
    dt = time.perf_counter() - t0
    t, _, _, _ = oracle.grid(w.seq)
    n_int = len(t) - 1
    stride = STATE_STRIDE[name]
    out = {"input_sha256": np.array(input_sha256(w)), "workload": np.array(w.name),
           "n_spins": np.int64(w.phantom.n), "n_intervals": np.int64(n_int),
           "oracle_seconds": np.float64(dt), "oracle_threads": np.int64(cores),
           "state_stride": np.int64(stride),
           "Mxy": mxy[::stride].astype(np.complex64), "Mz": mz[::stride].astype(np.float32)}
    if name == "5b":
        cols = columns_5b(sig.shape[1])
        out["columns"] = cols
        out["signal"] = np.ascontiguousarray(sig[:, cols]).astype(np.complex64)
    elif name == "4":
        out["signal"] = sig.astype(np.complex128)
    else:
        out["signal"] = sig.astype(np.complex64)
    np.savez_compressed(golden_path(name), **out)
    print(f"config {name}: {w.phantom.n} spins x {n_int} intervals, whole oracle in {dt:.1f} s on {cores} threads "
          f"({w.phantom.n * n_int / dt:.3e} spin*steps/s) -> {golden_path(name)} "
          f"({os.path.getsize(golden_path(name)) / 1e6:.1f} MB)", flush=True)


if __name__ == "__main__":
    for nm in (sys.argv[1:] or ["4", "5", "5b"]):
        if nm not in STATE_STRIDE:
            raise SystemExit(f"unknown config {nm!r}: choose from 4, 5, 5b")
        make(nm)
