"""Thin ctypes binding of libbloch_b200.so (include/bloch.h): argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels / host planner.  PyTorch is used for
device memory and streams only.  There is NO CPU fallback: importing this module without the built
extension raises, and nothing here imports ``oracle``.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libbloch_b200.so")

PHASE_AUTO, PHASE_FP32, PHASE_FP64 = 0, 1, 2
OUT_SUM_ALL, OUT_PER_SPIN, OUT_GROUPED = 0, 1, 2
_PHASE = {"auto": PHASE_AUTO, "fp32": PHASE_FP32, "fp64": PHASE_FP64}
_OUT = {"sum": OUT_SUM_ALL, "per_spin": OUT_PER_SPIN, "grouped": OUT_GROUPED}
MOTION_NONE, MOTION_LINEAR, MOTION_WAVEFORM = 0, 1, 2
_MOTION = {"none": MOTION_NONE, "linear": MOTION_LINEAR, "waveform": MOTION_WAVEFORM}

_dp = C.POINTER(C.c_double)
_fp = C.c_void_p  # float* (host or device) passed as an address


class bloch_scanner(C.Structure):
    _fields_ = [("gamma", C.c_double), ("B0", C.c_double), ("G_max", C.c_double), ("S_max", C.c_double)]


class bloch_sequence(C.Structure):
    _fields_ = [("g_t", _dp * 3), ("g_v", _dp * 3), ("g_n", C.c_int64 * 3),
                ("rf_t", _dp), ("rf_dt", _dp), ("rf_re", _dp), ("rf_im", _dp), ("rf_n", C.c_int64),
                ("adc_t", _dp), ("adc_n", C.c_int64), ("t_end", C.c_double)]


class bloch_sim_params(C.Structure):
    _fields_ = [("dt_max", C.c_double), ("dt_rf_max", C.c_double), ("max_block_points", C.c_int64),
                ("phase_mode", C.c_int32), ("output_mode", C.c_int32), ("motion_mode", C.c_int32),
                ("group_size", C.c_int32), ("max_extent_m", C.c_double), ("max_offres_hz", C.c_double),
                ("max_speed_mps", C.c_double), ("motion_t", _dp), ("motion_u", _dp), ("motion_n", C.c_int64)]


class bloch_plan_info(C.Structure):
    _fields_ = [("n_intervals", C.c_int64), ("n_rf_steps", C.c_int64), ("n_adc", C.c_int64),
                ("n_blocks", C.c_int64), ("n_rf_blocks", C.c_int64), ("n_eval_points", C.c_int64),
                ("n_launches", C.c_int64), ("table_bytes", C.c_int64), ("max_block_adc", C.c_int64),
                ("phase_mode", C.c_int32), ("output_mode", C.c_int32), ("motion_mode", C.c_int32),
                ("group_size", C.c_int32), ("phase_mode_requested", C.c_int32), ("path", C.c_int32),
                ("max_extent_m", C.c_double), ("max_offres_hz", C.c_double), ("max_speed_mps", C.c_double),
                ("worst_turns", C.c_double), ("options", C.c_int32 * 16)]


# BLOCH_OPT_* keys of bloch_plan_set_option, in enum order
OPTIONS = ("signal_lin", "signal_p", "signal_fixed_cta", "signal_ctas_per_sm", "rf_threads", "rf_spins", "coil_tc",
           "seq_sig_extra", "seq_sig_base", "seq_items_x4", "rf_const")
STATUS_BAD_RELAXATION, STATUS_NONFINITE, STATUS_PHASE_RANGE = 1, 2, 4

EXPORTS = ["bloch_version", "bloch_strerror", "bloch_last_error", "bloch_plan_create", "bloch_plan_destroy",
           "bloch_plan_get_info", "bloch_plan_workspace_bytes", "bloch_plan_upload", "bloch_simulate",
           "bloch_simulate_motion", "bloch_simulate_host_scratch_bytes", "bloch_simulate_host",
           "bloch_simulate_host_motion", "bloch_plan_set_profiling",
           "bloch_plan_last_timing", "bloch_plan_last_launches", "bloch_plan_set_path", "bloch_plan_uses_fused",
           "bloch_plan_workspace_bytes_coils", "bloch_simulate_coils", "bloch_simulate_host_coils_scratch_bytes",
           "bloch_simulate_host_coils", "bloch_plan_set_option", "bloch_plan_get_option", "bloch_plan_status",
           "bloch_plan_last_kernel", "bloch_simulate_coils_motion", "bloch_simulate_host_coils_motion", "bloch_sequence_write",
           "bloch_sequence_read", "bloch_sequence_file_get", "bloch_sequence_file_free", "bloch_signal_write",
           "bloch_signal_read", "bloch_plan_host_tables", "bloch_simulate_static", "bloch_microbench"]


def _load():
    if not os.path.exists(_SO):
        raise ImportError(f"{_SO} is missing: build it with `python -m paper_2301_02702_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(_SO)
    vp, i64, sz = C.c_void_p, C.c_int64, C.c_size_t
    lib.bloch_version.restype = C.c_int
    lib.bloch_strerror.restype = C.c_char_p
    lib.bloch_strerror.argtypes = [C.c_int]
    lib.bloch_last_error.restype = C.c_char_p
    lib.bloch_plan_create.argtypes = [C.POINTER(bloch_scanner), C.POINTER(bloch_sequence),
                                      C.POINTER(bloch_sim_params), C.POINTER(vp)]
    lib.bloch_plan_destroy.argtypes = [vp]
    lib.bloch_plan_get_info.argtypes = [vp, C.POINTER(bloch_plan_info)]
    lib.bloch_plan_workspace_bytes.argtypes = [vp, i64, C.POINTER(sz)]
    lib.bloch_plan_upload.argtypes = [vp, vp, sz, vp]
    sim_args = [vp, i64] + [_fp] * 7 + [_fp, _fp, C.c_int, _fp, vp, sz, vp]
    lib.bloch_simulate.argtypes = sim_args
    lib.bloch_simulate_static.argtypes = [vp, i64] + [_fp] * 7 + [_fp, _fp, C.c_int, _fp, vp]
    lib.bloch_simulate_host_scratch_bytes.argtypes = [vp, i64, C.POINTER(sz)]
    lib.bloch_simulate_host.argtypes = sim_args
    mo_args = [vp, i64] + [_fp] * 10 + [_fp, _fp, C.c_int, _fp, vp, sz, vp]
    lib.bloch_simulate_motion.argtypes = mo_args
    lib.bloch_simulate_host_motion.argtypes = mo_args
    lib.bloch_plan_workspace_bytes_coils.argtypes = [vp, i64, C.c_int, C.POINTER(sz)]
    lib.bloch_simulate_coils.argtypes = [vp, i64] + [_fp] * 7 + [C.c_int, _fp, _fp, _fp, C.c_int, _fp, vp, sz, vp]
    lib.bloch_simulate_host_coils_scratch_bytes.argtypes = [vp, i64, C.c_int, C.POINTER(sz)]
    lib.bloch_simulate_host_coils.argtypes = lib.bloch_simulate_coils.argtypes
    lib.bloch_simulate_coils_motion.argtypes = [vp, i64] + [_fp] * 10 + [C.c_int, _fp, _fp, _fp, C.c_int, _fp, vp, sz, vp]
    lib.bloch_simulate_host_coils_motion.argtypes = lib.bloch_simulate_coils_motion.argtypes
    lib.bloch_plan_set_profiling.argtypes = [vp, C.c_int]
    lib.bloch_plan_last_timing.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(i64)]
    lib.bloch_plan_last_launches.argtypes = [vp, C.POINTER(i64)]
    lib.bloch_plan_last_kernel.argtypes = [vp, C.c_int, C.c_char_p, sz, C.POINTER(i64), C.POINTER(C.c_int)]
    lib.bloch_plan_set_path.argtypes = [vp, C.c_int]
    lib.bloch_plan_uses_fused.argtypes = [vp, i64, C.POINTER(C.c_int)]
    lib.bloch_plan_set_option.argtypes = [vp, C.c_int, C.c_int]
    lib.bloch_plan_get_option.argtypes = [vp, C.c_int, C.POINTER(C.c_int)]
    lib.bloch_plan_status.argtypes = [vp, vp, C.POINTER(C.c_int)]
    lib.bloch_microbench.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double), vp]
    lib.bloch_plan_host_tables.argtypes = [vp, C.POINTER(vp), C.POINTER(sz)]
    lib.bloch_sequence_write.argtypes = [C.c_char_p, C.POINTER(bloch_scanner), C.POINTER(bloch_sequence)]
    lib.bloch_sequence_read.argtypes = [C.c_char_p, C.POINTER(vp)]
    lib.bloch_sequence_file_get.argtypes = [vp, C.POINTER(bloch_scanner), C.POINTER(bloch_sequence)]
    lib.bloch_sequence_file_free.argtypes = [vp]
    lib.bloch_signal_write.argtypes = [C.c_char_p, _fp, i64, i64, _dp]
    lib.bloch_signal_read.argtypes = [C.c_char_p, _fp, i64, C.POINTER(i64), C.POINTER(i64), _dp]
    for name in EXPORTS:
        if name not in ("bloch_strerror", "bloch_last_error"):
            getattr(lib, name).restype = C.c_int
    return lib


_lib = _load()


class BlochError(RuntimeError):
    def __init__(self, code: int):
        self.code = code
        detail = _lib.bloch_last_error().decode()
        super().__init__(f"{_lib.bloch_strerror(code).decode()} ({code}): {detail}")


def _check(rc: int):
    if rc != 0:
        raise BlochError(rc)


# ---- same-name wrappers (marshalling only) ------------------------------------------------------
def bloch_version() -> int:
    return _lib.bloch_version()


def bloch_strerror(code: int) -> str:
    return _lib.bloch_strerror(code).decode()


def bloch_last_error() -> str:
    return _lib.bloch_last_error().decode()


def _darr(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def _c_sequence(seq, keep):
    cs = bloch_sequence()
    for a in range(3):
        t, tp = _darr(seq.g_t[a]); v, vp_ = _darr(seq.g_v[a])
        if t.shape != v.shape:
            raise ValueError("g_t / g_v length mismatch")
        keep += [t, v]
        cs.g_t[a], cs.g_v[a], cs.g_n[a] = tp, vp_, t.shape[0]
    rt, cs.rf_t = _darr(seq.rf_t); rd, cs.rf_dt = _darr(seq.rf_dt)
    rr, cs.rf_re = _darr(seq.rf_re); ri, cs.rf_im = _darr(seq.rf_im)
    if not (rt.shape == rd.shape == rr.shape == ri.shape):
        raise ValueError("RF array length mismatch")
    ad, cs.adc_t = _darr(seq.adc_t)
    keep += [rt, rd, rr, ri, ad]
    cs.rf_n, cs.adc_n, cs.t_end = rt.shape[0], ad.shape[0], float(seq.t_end)
    return cs


def bloch_sequence_write(path: str, seq, *, gamma: float = 0.0, B0: float = 0.0, G_max: float = 0.0, S_max: float = 0.0):
    """Writes scanner + sequence to the library's own text container (bit-exact; NOT Pulseq)."""
    keep = []
    cs = _c_sequence(seq, keep)
    sc = bloch_scanner(float(gamma), float(B0), float(G_max), float(S_max))
    _check(_lib.bloch_sequence_write(os.fsencode(path), C.byref(sc), C.byref(cs)))


def bloch_sequence_read(path: str):
    """-> (scanner dict, sequence object with numpy copies of g_t, g_v, rf_t, rf_dt, rf_re, rf_im, adc_t, t_end)."""
    from types import SimpleNamespace
    h = C.c_void_p()
    _check(_lib.bloch_sequence_read(os.fsencode(path), C.byref(h)))
    try:
        sc, cs = bloch_scanner(), bloch_sequence()
        _check(_lib.bloch_sequence_file_get(h, C.byref(sc), C.byref(cs)))

        def arr(p, n):
            return np.ctypeslib.as_array(p, shape=(n,)).copy() if n else np.zeros(0)
        seq = SimpleNamespace(g_t=[arr(cs.g_t[a], cs.g_n[a]) for a in range(3)],
                              g_v=[arr(cs.g_v[a], cs.g_n[a]) for a in range(3)],
                              rf_t=arr(cs.rf_t, cs.rf_n), rf_dt=arr(cs.rf_dt, cs.rf_n), rf_re=arr(cs.rf_re, cs.rf_n),
                              rf_im=arr(cs.rf_im, cs.rf_n), adc_t=arr(cs.adc_t, cs.adc_n), t_end=float(cs.t_end))
        scanner = dict(gamma=sc.gamma, B0=sc.B0, G_max=sc.G_max, S_max=sc.S_max)
    finally:
        _lib.bloch_sequence_file_free(h)
    return scanner, seq


def bloch_signal_write(path: str, signal, adc_t=None):
    """signal: complex64 numpy array [n_adc] or [rows, n_adc]; adc_t optional float64 [n_adc]."""
    sig = np.ascontiguousarray(signal, dtype=np.complex64)
    rows, n_adc = (1, sig.shape[0]) if sig.ndim == 1 else (sig.shape[0], sig.shape[1])
    t = None if adc_t is None else np.ascontiguousarray(adc_t, dtype=np.float64)
    if t is not None and t.shape != (n_adc,):
        raise ValueError("adc_t must hold n_adc times")
    _check(_lib.bloch_signal_write(os.fsencode(path), sig.ctypes.data, rows, n_adc,
                                   None if t is None else t.ctypes.data_as(_dp)))


def bloch_signal_read(path: str):
    """-> (complex64 [rows, n_adc], adc_t float64 [n_adc])."""
    rows, n_adc = C.c_int64(), C.c_int64()
    _check(_lib.bloch_signal_read(os.fsencode(path), None, 0, C.byref(rows), C.byref(n_adc), None))
    sig = np.zeros((rows.value, n_adc.value), dtype=np.complex64)
    t = np.zeros(n_adc.value, dtype=np.float64)
    _check(_lib.bloch_signal_read(os.fsencode(path), sig.ctypes.data, sig.size, C.byref(rows), C.byref(n_adc),
                                  t.ctypes.data_as(_dp)))
    return sig, t


def bloch_plan_create(seq, *, gamma: float = 0.0, dt_rf_max: float | None = None, dt_max: float = 0.0,
                      max_block_points: int = 0, phase_mode="auto", output_mode="sum", motion="none",
                      group_size: int = 0, G_max: float = 0.0, S_max: float = 0.0, B0: float = 0.0,
                      max_extent_m: float = 0.0, max_offres_hz: float = 0.0, max_speed_mps: float = 0.0,
                      waveform=None) -> int:
    """G_max [T/m], S_max [T/m/s]: scanner limits the gradient waveforms are checked against when > 0.
    max_extent_m / max_offres_hz / max_speed_mps: extents of the phantoms the plan will see (bloch_sim_params).
    waveform: (t, u) vertex arrays of the shared motion waveform for motion="waveform" (x(t) = x + a u(t)).
    seq: object with g_t, g_v (3 arrays each), rf_t, rf_dt, rf_re, rf_im, adc_t, t_end[, dt_rf_max].
    Returns the opaque plan handle (an integer address)."""
    keep = []
    cs = _c_sequence(seq, keep)
    if dt_rf_max is None:
        dt_rf_max = float(getattr(seq, "dt_rf_max", 0.0))
    sc = bloch_scanner(float(gamma), float(B0), float(G_max), float(S_max))
    pm = _PHASE[phase_mode] if isinstance(phase_mode, str) else int(phase_mode)
    om = _OUT[output_mode] if isinstance(output_mode, str) else int(output_mode)
    mm = _MOTION[motion] if isinstance(motion, str) else int(motion)
    sp = bloch_sim_params(float(dt_max), float(dt_rf_max), int(max_block_points), pm, om, mm, int(group_size),
                          float(max_extent_m), float(max_offres_hz), float(max_speed_mps))
    if waveform is not None:
        wt, sp.motion_t = _darr(waveform[0]); wu, sp.motion_u = _darr(waveform[1])
        if wt.shape != wu.shape or wt.ndim != 1:
            raise ValueError("waveform must be two equally long 1-D arrays (t, u)")
        keep += [wt, wu]
        sp.motion_n = wt.shape[0]
    h = C.c_void_p()
    _check(_lib.bloch_plan_create(C.byref(sc), C.byref(cs), C.byref(sp), C.byref(h)))
    return h.value


def bloch_plan_destroy(plan: int):
    _check(_lib.bloch_plan_destroy(plan))


def bloch_plan_get_info(plan: int) -> dict:
    inf = bloch_plan_info()
    _check(_lib.bloch_plan_get_info(plan, C.byref(inf)))
    out = {}
    for k, tp in bloch_plan_info._fields_:
        v = getattr(inf, k)
        if k == "options":
            out[k] = {name: int(v[i]) for i, name in enumerate(OPTIONS)}
        else:
            out[k] = float(v) if tp is C.c_double else int(v)
    return out


def bloch_plan_host_tables(plan: int) -> bytes:
    """A copy of the plan's table image (what bloch_plan_upload sends to the device)."""
    ptr, n = C.c_void_p(), C.c_size_t()
    _check(_lib.bloch_plan_host_tables(plan, C.byref(ptr), C.byref(n)))
    return C.string_at(ptr.value, n.value)


def bloch_plan_workspace_bytes(plan: int, n_spins: int) -> int:
    out = C.c_size_t()
    _check(_lib.bloch_plan_workspace_bytes(plan, n_spins, C.byref(out)))
    return int(out.value)


def bloch_plan_upload(plan: int, d_tables_ptr: int, nbytes: int, stream: int = 0):
    _check(_lib.bloch_plan_upload(plan, d_tables_ptr, nbytes, stream))


def bloch_simulate(plan: int, n_spins: int, x, y, z, M0, T1, T2, dw, Mxy, Mz, init_equilibrium: bool,
                   signal, workspace, workspace_bytes: int, stream: int = 0):
    """All array arguments are raw DEVICE addresses (ints) or None."""
    _check(_lib.bloch_simulate(plan, n_spins, x, y, z, M0, T1, T2, dw, Mxy, Mz, int(bool(init_equilibrium)),
                               signal, workspace, workspace_bytes, stream))


STATIC_WORKSPACE_BYTES = 32 << 20  # BLOCH_STATIC_WORKSPACE_BYTES of include/bloch.h


def bloch_simulate_static(plan: int, n_spins: int, x, y, z, M0, T1, T2, dw, Mxy, Mz, init_equilibrium: bool,
                          signal, stream: int = 0):
    """bloch_simulate on the library's own static device workspace (allocates nothing; static plans whose workspace
    is at most STATIC_WORKSPACE_BYTES).  All array arguments are raw DEVICE addresses (ints) or None."""
    _check(_lib.bloch_simulate_static(plan, n_spins, x, y, z, M0, T1, T2, dw, Mxy, Mz, int(bool(init_equilibrium)),
                                      signal, stream))


def bloch_simulate_motion(plan: int, n_spins: int, x, y, z, M0, T1, T2, dw, vx, vy, vz, Mxy, Mz,
                          init_equilibrium: bool, signal, workspace, workspace_bytes: int, stream: int = 0):
    """bloch_simulate with per-spin velocities (raw DEVICE addresses or None for all three)."""
    _check(_lib.bloch_simulate_motion(plan, n_spins, x, y, z, M0, T1, T2, dw, vx, vy, vz, Mxy, Mz,
                                      int(bool(init_equilibrium)), signal, workspace, workspace_bytes, stream))


def bloch_plan_workspace_bytes_coils(plan: int, n_spins: int, n_coils: int) -> int:
    out = C.c_size_t()
    _check(_lib.bloch_plan_workspace_bytes_coils(plan, n_spins, n_coils, C.byref(out)))
    return int(out.value)


def bloch_simulate_coils(plan: int, n_spins: int, x, y, z, M0, T1, T2, dw, n_coils: int, coil, Mxy, Mz,
                         init_equilibrium: bool, signal, workspace, workspace_bytes: int, stream: int = 0):
    """bloch_simulate with n_coils receive coils: coil = DEVICE address of float2 [n_coils][n_spins], signal =
    DEVICE address of float2 [n_coils][n_adc]."""
    _check(_lib.bloch_simulate_coils(plan, n_spins, x, y, z, M0, T1, T2, dw, n_coils, coil, Mxy, Mz,
                                     int(bool(init_equilibrium)), signal, workspace, workspace_bytes, stream))


def bloch_simulate_coils_motion(plan: int, n_spins: int, x, y, z, M0, T1, T2, dw, vx, vy, vz, n_coils: int, coil, Mxy, Mz,
                                init_equilibrium: bool, signal, workspace, workspace_bytes: int, stream: int = 0):
    """bloch_simulate_coils for moving spins (motion plans); vx, vy, vz raw DEVICE addresses or None for all three."""
    _check(_lib.bloch_simulate_coils_motion(plan, n_spins, x, y, z, M0, T1, T2, dw, vx, vy, vz, n_coils, coil, Mxy, Mz,
                                            int(bool(init_equilibrium)), signal, workspace, workspace_bytes, stream))


def bloch_simulate_host_coils_motion(plan: int, n_spins: int, x, y, z, M0, T1, T2, dw, vx, vy, vz, n_coils: int, coil, Mxy,
                                     Mz, init_equilibrium: bool, signal, scratch, scratch_bytes: int, stream: int = 0):
    """bloch_simulate_coils_motion with HOST phantom / velocity / coil / state / signal addresses."""
    _check(_lib.bloch_simulate_host_coils_motion(plan, n_spins, x, y, z, M0, T1, T2, dw, vx, vy, vz, n_coils, coil, Mxy,
                                                 Mz, int(bool(init_equilibrium)), signal, scratch, scratch_bytes, stream))


def bloch_simulate_host_coils_scratch_bytes(plan: int, n_spins: int, n_coils: int) -> int:
    out = C.c_size_t()
    _check(_lib.bloch_simulate_host_coils_scratch_bytes(plan, n_spins, n_coils, C.byref(out)))
    return int(out.value)


def bloch_simulate_host_coils(plan: int, n_spins: int, x, y, z, M0, T1, T2, dw, n_coils: int, coil, Mxy, Mz,
                              init_equilibrium: bool, signal, scratch, scratch_bytes: int, stream: int = 0):
    """bloch_simulate_coils with HOST phantom / coil / state / signal addresses; scratch is a device address."""
    _check(_lib.bloch_simulate_host_coils(plan, n_spins, x, y, z, M0, T1, T2, dw, n_coils, coil, Mxy, Mz,
                                          int(bool(init_equilibrium)), signal, scratch, scratch_bytes, stream))


def bloch_simulate_host_motion(plan: int, n_spins: int, x, y, z, M0, T1, T2, dw, vx, vy, vz, Mxy, Mz,
                               init_equilibrium: bool, signal, scratch, scratch_bytes: int, stream: int = 0):
    """bloch_simulate_host with per-spin velocities (raw HOST addresses or None for all three)."""
    _check(_lib.bloch_simulate_host_motion(plan, n_spins, x, y, z, M0, T1, T2, dw, vx, vy, vz, Mxy, Mz,
                                           int(bool(init_equilibrium)), signal, scratch, scratch_bytes, stream))


def bloch_simulate_host_scratch_bytes(plan: int, n_spins: int) -> int:
    out = C.c_size_t()
    _check(_lib.bloch_simulate_host_scratch_bytes(plan, n_spins, C.byref(out)))
    return int(out.value)


def bloch_simulate_host(plan: int, n_spins: int, x, y, z, M0, T1, T2, dw, Mxy, Mz, init_equilibrium: bool,
                        signal, scratch, scratch_bytes: int, stream: int = 0):
    """Phantom / state / signal arguments are raw HOST addresses (ints) or None; scratch is a device address."""
    _check(_lib.bloch_simulate_host(plan, n_spins, x, y, z, M0, T1, T2, dw, Mxy, Mz,
                                    int(bool(init_equilibrium)), signal, scratch, scratch_bytes, stream))


def bloch_plan_set_profiling(plan: int, enable: bool):
    _check(_lib.bloch_plan_set_profiling(plan, int(bool(enable))))


KINDS = ("other", "rf", "signal", "reduce", "fused")   # BLOCH_KIND_*
PATHS = {"auto": 0, "per_block": 1, "fused": 2}       # BLOCH_PATH_*


def bloch_plan_set_path(plan: int, path):
    _check(_lib.bloch_plan_set_path(plan, PATHS[path] if isinstance(path, str) else int(path)))


def bloch_plan_set_option(plan: int, key, value: int):
    """key: a BLOCH_OPT_* integer or its name in OPTIONS."""
    _check(_lib.bloch_plan_set_option(plan, OPTIONS.index(key) if isinstance(key, str) else int(key), int(value)))


def bloch_plan_get_option(plan: int, key) -> int:
    out = C.c_int()
    _check(_lib.bloch_plan_get_option(plan, OPTIONS.index(key) if isinstance(key, str) else int(key), C.byref(out)))
    return int(out.value)


def bloch_plan_status(plan: int, stream: int = 0) -> int:
    """Synchronises `stream`; raises BlochError (BLOCH_EINVAL / BLOCH_ERANGE) when the last simulation's phantom was
    invalid or outside the plan's phase range, else returns the (zero) status flags."""
    flags = C.c_int()
    _check(_lib.bloch_plan_status(plan, stream, C.byref(flags)))
    return int(flags.value)


def bloch_plan_uses_fused(plan: int, n_spins: int) -> bool:
    out = C.c_int()
    _check(_lib.bloch_plan_uses_fused(plan, n_spins, C.byref(out)))
    return bool(out.value)


def bloch_plan_last_timing(plan: int) -> dict:
    ms = (C.c_float * len(KINDS))()
    cnt = (C.c_int64 * len(KINDS))()
    _check(_lib.bloch_plan_last_timing(plan, ms, cnt))
    return {"ms": {k: float(ms[i]) for i, k in enumerate(KINDS)},
            "launches": {k: int(cnt[i]) for i, k in enumerate(KINDS)}}


def bloch_plan_last_launches(plan: int) -> int:
    out = C.c_int64()
    _check(_lib.bloch_plan_last_launches(plan, C.byref(out)))
    return int(out.value)


def bloch_plan_last_kernel(plan: int, kind) -> dict:
    """kind: BLOCH_KIND_* integer or its name in KINDS -> {"name", "grid", "block"} of that kind's largest launch."""
    buf = C.create_string_buffer(64)
    grid, block = C.c_int64(), C.c_int()
    _check(_lib.bloch_plan_last_kernel(plan, KINDS.index(kind) if isinstance(kind, str) else int(kind), buf, 64,
                                       C.byref(grid), C.byref(block)))
    return {"name": buf.value.decode(), "grid": int(grid.value), "block": int(block.value)}


def bloch_microbench(kind: int, iters: int = 4096, stream: int = 0) -> float:
    out = C.c_double()
    _check(_lib.bloch_microbench(kind, iters, C.byref(out), stream))
    return float(out.value)


# ---- convenience object: owns the handle and the torch buffers ------------------------------------
class Plan:
    """Owns a bloch_plan handle plus the caller-side device buffers (torch tensors)."""

    def __init__(self, seq, path="auto", options=None, **kw):
        """options: {name in OPTIONS: value} passed to bloch_plan_set_option (kernel selection is plan state)."""
        self.handle = bloch_plan_create(seq, **kw)
        bloch_plan_set_path(self.handle, path)
        for k, v in (options or {}).items():
            bloch_plan_set_option(self.handle, k, v)
        self.info = bloch_plan_get_info(self.handle)
        self._tables = None
        self._ws = None
        self._scratch = None

    def close(self):
        if getattr(self, "handle", None):
            bloch_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key, value):
        bloch_plan_set_option(self.handle, key, value)
        self.info = bloch_plan_get_info(self.handle)
        self._ws = None     # launch shapes enter the workspace size
        return self

    def status(self):
        """Synchronises the current stream and raises if the last simulate() met an invalid phantom (bad T1 / T2,
        non-finite values) or one outside the plan's phase range."""
        return bloch_plan_status(self.handle, self._stream())

    @staticmethod
    def _check_out(t, numel, dtypes, what):
        import torch
        if t is None:
            return
        assert isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous(), f"{what}: contiguous CUDA tensor needed"
        assert t.dtype in dtypes, f"{what}: dtype {t.dtype} not in {dtypes}"
        n = t.numel() * (2 if t.dtype == torch.complex64 else 1)
        assert n == numel, f"{what}: {n} fp32 values given, {numel} expected"

    def _signal_shape(self, n):
        n_adc, mode = self.info["n_adc"], self.info["output_mode"]
        if mode == OUT_PER_SPIN:
            return (n, n_adc)
        if mode == OUT_GROUPED:
            return (n // max(1, self.info["group_size"]), n_adc)
        return (n_adc,)

    @staticmethod
    def _stream():
        import torch
        return int(torch.cuda.current_stream().cuda_stream)

    def upload(self):
        import torch
        self._tables = torch.empty(max(self.info["table_bytes"], 256), dtype=torch.uint8, device="cuda")
        bloch_plan_upload(self.handle, self._tables.data_ptr(), self._tables.numel(), self._stream())
        return self

    def _workspace(self, n, n_coils=0):
        import torch
        need = max(bloch_plan_workspace_bytes_coils(self.handle, n, n_coils), 256)
        if self._ws is None or self._ws.numel() < need:
            self._ws = torch.empty(need, dtype=torch.uint8, device="cuda")
        return self._ws

    def simulate(self, x, y, z, M0, T1, T2, dw, Mxy=None, Mz=None, init_equilibrium=True, signal=None,
                 velocity=None, coils=None):
        """Device path: torch float32 CUDA tensors in, complex64 signal tensor out (asynchronous).
        velocity: optional (vx, vy, vz) float32 CUDA tensors (plan created with motion="linear").
        coils: optional complex64 CUDA tensor [n_coils, n_spins] of receive sensitivities; the signal is then
        [n_coils, n_adc] (bloch_simulate_coils)."""
        import torch
        if self._tables is None:
            self.upload()
        n = int(x.numel())
        for t in (x, y, z, M0, T1, T2, dw):
            assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.numel() == n
        n_adc = self.info["n_adc"]
        shape = self._signal_shape(n)
        # the C side only sees raw pointers: wrong sizes or dtypes would be out-of-bounds device writes
        self._check_out(Mxy, 2 * n, (torch.float32, torch.complex64), "Mxy")
        self._check_out(Mz, n, (torch.float32,), "Mz")
        n_rows = int(coils.shape[0]) if coils is not None and coils.dim() == 2 else int(np.prod(shape[:-1]))
        self._check_out(signal, 2 * n_rows * n_adc, (torch.complex64,), "signal")
        if coils is not None:
            assert coils.is_cuda and coils.dtype == torch.complex64 and coils.is_contiguous() and \
                coils.dim() == 2 and coils.shape[1] == n
            n_coils = int(coils.shape[0])
            if signal is None:
                signal = torch.empty((n_coils, n_adc), dtype=torch.complex64, device="cuda")
            ws = self._workspace(n, n_coils)
            vp = [None, None, None]
            if velocity is not None:
                for t in velocity:
                    assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.numel() == n
                vp = [t.data_ptr() for t in velocity]
            bloch_simulate_coils_motion(self.handle, n, x.data_ptr(), y.data_ptr(), z.data_ptr(), M0.data_ptr(),
                                        T1.data_ptr(), T2.data_ptr(), dw.data_ptr(), *vp, n_coils, coils.data_ptr(),
                                        None if Mxy is None else Mxy.data_ptr(), None if Mz is None else Mz.data_ptr(),
                                        init_equilibrium, signal.data_ptr() if signal.numel() else None,
                                        ws.data_ptr(), ws.numel(), self._stream())
            return signal
        if signal is None:
            signal = torch.empty(shape, dtype=torch.complex64, device="cuda")
        ws = self._workspace(n)
        vp = [None, None, None]
        if velocity is not None:
            for t in velocity:
                assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.numel() == n
            vp = [t.data_ptr() for t in velocity]
        bloch_simulate_motion(self.handle, n, x.data_ptr(), y.data_ptr(), z.data_ptr(), M0.data_ptr(), T1.data_ptr(),
                              T2.data_ptr(), dw.data_ptr(), *vp,
                              None if Mxy is None else Mxy.data_ptr(), None if Mz is None else Mz.data_ptr(),
                              init_equilibrium, signal.data_ptr() if signal.numel() else None,
                              ws.data_ptr(), ws.numel(), self._stream())
        return signal

    def simulate_static(self, x, y, z, M0, T1, T2, dw, signal, Mxy=None, Mz=None, init_equilibrium=True):
        """bloch_simulate_static: as simulate(), but the workspace is the library's static device array and NOTHING is
        allocated here either -- `signal` (complex64 CUDA tensor of the plan's output shape) must be passed in.  Calls
        whose GPU work overlaps race on the shared array: keep them on one stream."""
        import torch
        if self._tables is None:
            raise RuntimeError("upload() the plan's tables first (simulate_static allocates nothing)")
        n = int(x.numel())
        for t in (x, y, z, M0, T1, T2, dw):
            assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.numel() == n
        n_rows = int(np.prod(self._signal_shape(n)[:-1]))
        assert signal is not None, "simulate_static writes into a caller tensor"
        self._check_out(Mxy, 2 * n, (torch.float32, torch.complex64), "Mxy")
        self._check_out(Mz, n, (torch.float32,), "Mz")
        self._check_out(signal, 2 * n_rows * self.info["n_adc"], (torch.complex64,), "signal")
        bloch_simulate_static(self.handle, n, x.data_ptr(), y.data_ptr(), z.data_ptr(), M0.data_ptr(), T1.data_ptr(),
                              T2.data_ptr(), dw.data_ptr(), None if Mxy is None else Mxy.data_ptr(),
                              None if Mz is None else Mz.data_ptr(), init_equilibrium,
                              signal.data_ptr() if signal.numel() else None, self._stream())
        return signal

    def simulate_host(self, x, y, z, M0, T1, T2, dw, Mxy=None, Mz=None, init_equilibrium=True, signal=None,
                      velocity=None, coils=None):
        """End-to-end path: numpy float32 HOST arrays in, numpy complex64 signal out (synchronous)."""
        import torch
        if self._tables is None:
            self.upload()
        arrs = [np.ascontiguousarray(a, dtype=np.float32) for a in (x, y, z, M0, T1, T2, dw)]
        n = int(arrs[0].shape[0])
        assert all(a.shape == (n,) for a in arrs), "phantom arrays must all hold n_spins values"
        n_adc = self.info["n_adc"]
        shape = self._signal_shape(n)
        n_rows = int(np.shape(coils)[0]) if coils is not None else int(np.prod(shape[:-1]))
        for a, cnt, dts, what in ((Mxy, 2 * n, (np.float32, np.complex64), "Mxy"), (Mz, n, (np.float32,), "Mz"),
                                  (signal, 2 * n_rows * n_adc, (np.complex64,), "signal")):
            if a is not None:
                assert isinstance(a, np.ndarray) and a.flags.c_contiguous and a.flags.writeable and \
                    a.dtype in dts, f"{what}: writable C-contiguous numpy array of dtype {dts} needed"
                assert a.size * (2 if a.dtype == np.complex64 else 1) == cnt, f"{what}: wrong size"
        if signal is None and coils is None:
            signal = np.empty(shape, dtype=np.complex64)
        if coils is not None:
            cw = np.ascontiguousarray(coils, dtype=np.complex64)
            assert cw.ndim == 2 and cw.shape[1] == n
            n_coils = int(cw.shape[0])
            hv = [None, None, None] if velocity is None else \
                [np.ascontiguousarray(a, dtype=np.float32) for a in velocity]
            if signal is None or signal.shape != (n_coils, n_adc):
                signal = np.empty((n_coils, n_adc), dtype=np.complex64)
            need = max(bloch_simulate_host_coils_scratch_bytes(self.handle, n, n_coils), 256)
            if self._scratch is None or self._scratch.numel() < need:
                self._scratch = torch.empty(need, dtype=torch.uint8, device="cuda")
            bloch_simulate_host_coils_motion(self.handle, n, *[a.ctypes.data for a in arrs],
                                             *[None if a is None else a.ctypes.data for a in hv], n_coils, cw.ctypes.data,
                                             None if Mxy is None else Mxy.ctypes.data, None if Mz is None else Mz.ctypes.data,
                                             init_equilibrium, signal.ctypes.data if signal.size else None,
                                             self._scratch.data_ptr(), self._scratch.numel(), self._stream())
            return signal
        need = max(bloch_simulate_host_scratch_bytes(self.handle, n), 256)
        if self._scratch is None or self._scratch.numel() < need:
            self._scratch = torch.empty(need, dtype=torch.uint8, device="cuda")
        vel = [None, None, None]
        if velocity is not None:
            vel = [np.ascontiguousarray(a, dtype=np.float32) for a in velocity]
        bloch_simulate_host_motion(self.handle, n, *[a.ctypes.data for a in arrs],
                                   *[None if a is None else a.ctypes.data for a in vel],
                                   None if Mxy is None else Mxy.ctypes.data, None if Mz is None else Mz.ctypes.data,
                                   init_equilibrium, signal.ctypes.data if signal.size else None,
                                   self._scratch.data_ptr(), self._scratch.numel(), self._stream())
        return signal


def phantom_to_device(ph):
    """Phantom (fp64 numpy, fp32-exact values) -> tuple of 7 float32 CUDA tensors."""
    import torch
    return tuple(torch.from_numpy(np.ascontiguousarray(getattr(ph, k), dtype=np.float32)).cuda()
                 for k in ("x", "y", "z", "M0", "T1", "T2", "dw"))
