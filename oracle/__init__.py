"""CPU fp64 oracle (TEST INFRASTRUCTURE ONLY -- see the header of bloch_ref.c).

ctypes wrapper around ``libbloch_ref.so`` built from ``oracle/bloch_ref.c`` with gcc.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs may import this
package.  It imports nothing from ``paper_2301_02702_b200`` (inputs are passed in as plain arrays or as
any object with the attribute names used below).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bloch_ref.c")
_SO = os.path.join(_HERE, "libbloch_ref.so")
_lib = None

GAMMA = 2.0 * np.pi * 42.58e6  # reading G4


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no fast-math, OpenMP over spins)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", _SRC, "-o", _SO, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        dp, i64 = C.POINTER(C.c_double), C.c_int64
        seq_args = [dp, dp, i64] * 3 + [dp, dp, dp, dp, i64, dp, i64, C.c_double, C.c_double]
        _lib.bloch_ref_simulate.restype = C.c_int
        _lib.bloch_ref_simulate.argtypes = ([C.c_double] + seq_args + [i64] + [dp] * 7 +
                                            [dp, dp, C.c_int, dp, C.c_int, C.c_int, C.c_int])
        _lib.bloch_ref_simulate_motion.restype = C.c_int
        _lib.bloch_ref_simulate_motion.argtypes = (_lib.bloch_ref_simulate.argtypes + [C.c_double, dp, dp, dp])
        _lib.bloch_ref_simulate_waveform.restype = C.c_int
        _lib.bloch_ref_simulate_waveform.argtypes = (_lib.bloch_ref_simulate_motion.argtypes + [dp, dp, i64])
        _lib.bloch_ref_grid.restype = i64
        _lib.bloch_ref_grid.argtypes = seq_args + [dp, dp, C.POINTER(C.c_uint8), C.POINTER(i64)]
        _lib.bloch_ref_grid_motion.restype = i64
        _lib.bloch_ref_grid_motion.argtypes = _lib.bloch_ref_grid.argtypes + [C.c_double]
        _lib.bloch_ref_grid_waveform.restype = i64
        _lib.bloch_ref_grid_waveform.argtypes = _lib.bloch_ref_grid_motion.argtypes + [dp, dp, i64, dp]
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _seq_args(seq, keep):
    args = []
    for a in range(3):
        t, tp = _d(seq.g_t[a]); v, vp = _d(seq.g_v[a])
        keep += [t, v]
        args += [tp, vp, C.c_int64(t.shape[0])]
    rt, rtp = _d(seq.rf_t); rd, rdp = _d(seq.rf_dt); rr, rrp = _d(seq.rf_re); ri, rip = _d(seq.rf_im)
    ad, adp = _d(seq.adc_t)
    keep += [rt, rd, rr, ri, ad]
    args += [rtp, rdp, rrp, rip, C.c_int64(rt.shape[0]), adp, C.c_int64(ad.shape[0]),
             C.c_double(seq.t_end), C.c_double(seq.dt_rf_max)]
    return args, int(ad.shape[0])


def simulate(phantom, seq, *, output_mode: str = "sum", state=None, return_state: bool = False,
             n_threads: int | None = None, gamma: float = GAMMA, force_excitation: bool = False,
             velocity=None, dt_max: float = 0.0, group_size: int = 0, coils=None, waveform=None):
    """Step-by-step fp64 Bloch integration (SURVEY.md 8(c) listing).

    phantom: object with fp64 arrays x, y, z, M0, T1, T2, dw.   seq: object with g_t, g_v (3 arrays each),
    rf_t, rf_dt, rf_re, rf_im, adc_t, t_end, dt_rf_max.
    velocity: optional (vx, vy, vz) fp64 arrays [m/s]: every spin moves as x(t) = x + v t;
    dt_max then refines every interval to at most dt_max (:180).
    waveform: optional (t, u) vertex arrays of a shared piecewise-linear motion waveform: every spin then moves as
    x(t) = x + velocity * u(t) (velocity = per-spin amplitude vectors; u held at its end values outside the vertices,
    which join the time grid); without it u(t) = t (reading M2; "motion field u(x, t)").
    Returns complex128 signal [n_adc] ("sum") or [n_spins, n_adc] ("per_spin"); with return_state also
    (Mxy complex128 [n_spins], Mz float64 [n_spins]).
    coils: optional complex [n_coils, n_spins] receive sensitivities at the spins (output_mode "sum" only):
    the signal becomes [n_coils, n_adc] (SURVEY.md 8(f) f2 "per-coil weights"; reading C1).
    """
    if coils is not None:
        # Reading C1 (the paper has no coils yet, :372 "straightforward to implement"): the standard receive
        # model S_c(t_j) = sum_i C_c(x_i) Mxy_i(t_j), C_c complex, no conjugation -- by definition the per-spin
        # signals weighted and added per coil.
        if output_mode != "sum":
            raise ValueError("coils need output_mode='sum'")
        Wc = np.asarray(coils, dtype=np.complex128)
        n_all = int(np.asarray(phantom.x).shape[0])
        if Wc.ndim != 2 or Wc.shape[1] != n_all:
            raise ValueError("coils must be [n_coils, n_spins]")
        res = simulate(phantom, seq, output_mode="per_spin", state=state, return_state=return_state,
                       n_threads=n_threads, gamma=gamma, force_excitation=force_excitation, velocity=velocity,
                       dt_max=dt_max, waveform=waveform)
        per = res[0] if return_state else res
        out = Wc @ per
        return (out,) + tuple(res[1:]) if return_state else out
    if output_mode == "grouped":
        # S[g][j] = sum of Mxy over the spins of group g (consecutive blocks of group_size
        # spins: an isochromat ensemble per voxel / dictionary entry) -- by definition the
        # per-spin signals added up group by group.
        n_all = int(np.asarray(phantom.x).shape[0])
        if group_size <= 0 or n_all % group_size:
            raise ValueError("group_size must be positive and divide the number of spins")
        res = simulate(phantom, seq, output_mode="per_spin", state=state, return_state=return_state,
                       n_threads=n_threads, gamma=gamma, force_excitation=force_excitation, velocity=velocity,
                       dt_max=dt_max, waveform=waveform)
        per = res[0] if return_state else res
        grouped = per.reshape(n_all // group_size, group_size, per.shape[1]).sum(axis=1)
        return (grouped,) + tuple(res[1:]) if return_state else grouped
    lib = _load()
    keep = []
    sargs, n_adc = _seq_args(seq, keep)
    n = int(np.asarray(phantom.x).shape[0])
    pa = []
    for name in ("x", "y", "z", "M0", "T1", "T2", "dw"):
        a, p = _d(getattr(phantom, name))
        keep.append(a)
        pa.append(p)
    mode = {"sum": 0, "per_spin": 1}[output_mode]
    if state is not None:
        mxy = np.ascontiguousarray(state[0], dtype=np.complex128).copy()
        mz = np.ascontiguousarray(state[1], dtype=np.float64).copy()
        use_state = 1
    else:
        mxy = np.zeros(n, dtype=np.complex128)
        mz = np.zeros(n, dtype=np.float64)
        use_state = 0
    sig = np.zeros((n, n_adc) if mode == 1 else (n_adc,), dtype=np.complex128)
    if n_threads is None:
        n_threads = os.cpu_count() or 1
    dp = C.POINTER(C.c_double)
    common = [C.c_double(gamma), *sargs, C.c_int64(n), *pa, mxy.ctypes.data_as(dp), mz.ctypes.data_as(dp),
              C.c_int(use_state), sig.ctypes.data_as(dp), C.c_int(mode), C.c_int(int(n_threads)),
              C.c_int(1 if force_excitation else 0)]
    if waveform is not None and velocity is None:
        raise ValueError("a motion waveform needs per-spin amplitudes (velocity=)")
    if velocity is None and not dt_max:
        rc = lib.bloch_ref_simulate(*common)
    else:
        va = [None, None, None]
        if velocity is not None:
            for k in range(3):
                a, pk = _d(np.broadcast_to(np.asarray(velocity[k], dtype=np.float64), (n,)))
                keep.append(a)
                va[k] = pk
        if waveform is None:
            rc = lib.bloch_ref_simulate_motion(*common, C.c_double(float(dt_max)), *va)
        else:
            wt, wtp = _d(waveform[0]); wu, wup = _d(waveform[1])
            if wt.shape != wu.shape or wt.ndim != 1 or wt.shape[0] < 1:
                raise ValueError("waveform must be two equally long 1-D arrays (t, u)")
            keep += [wt, wu]
            rc = lib.bloch_ref_simulate_waveform(*common, C.c_double(float(dt_max)), *va, wtp, wup,
                                                 C.c_int64(wt.shape[0]))
    if rc != 0:
        raise ValueError(f"bloch_ref_simulate failed with code {rc}")
    if return_state:
        return sig, mxy, mz
    return sig


def grid(seq, dt_max: float = 0.0, waveform=None):
    """The oracle's own discretisation: (t[n+1], G[n+1,3], rf[n] uint8, adc[n+1] int64); with a motion waveform
    (t, u) its vertices are points of the grid."""
    lib = _load()
    keep = []
    sargs, _ = _seq_args(seq, keep)
    null_d = C.POINTER(C.c_double)()
    wargs = [null_d, null_d, C.c_int64(0), null_d]
    if waveform is not None:
        wt, wtp = _d(waveform[0]); wu, wup = _d(waveform[1])
        keep += [wt, wu]
        wargs = [wtp, wup, C.c_int64(wt.shape[0]), null_d]
    n = lib.bloch_ref_grid_waveform(*sargs, null_d, null_d, C.POINTER(C.c_uint8)(), C.POINTER(C.c_int64)(),
                                    C.c_double(float(dt_max)), *wargs)
    if n < 0:
        raise ValueError(f"bloch_ref_grid failed with code {n}")
    t = np.zeros(n + 1); G = np.zeros((n + 1, 3)); rf = np.zeros(max(n, 1), dtype=np.uint8)
    adc = np.zeros(n + 1, dtype=np.int64)
    dp = C.POINTER(C.c_double)
    lib.bloch_ref_grid_waveform(*sargs, t.ctypes.data_as(dp), G.ctypes.data_as(dp),
                                rf.ctypes.data_as(C.POINTER(C.c_uint8)), adc.ctypes.data_as(C.POINTER(C.c_int64)),
                                C.c_double(float(dt_max)), *wargs)
    return t, G, rf[:n], adc
