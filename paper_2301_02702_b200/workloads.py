"""Seeded synthetic input generators (phantoms + pulse sequences) for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: it only *designs* inputs (spin property arrays, gradient vertices, RF samples, ADC times).
It imports neither the C-ABI binding nor anything under ``oracle/``.

Inputs stand in for the paper's workloads (EPI / spiral GRE on brain-like phantoms, PAPER.md:232-240;
slice-selective sinc + multi-shot spiral, :248; MRF, :268).  The BrainWeb / MRiLab phantoms the paper
used are not available here and are not reproduced; every array below is synthetic and seeded
(seed = 230102702 + config number).  Recipe: DESIGN.md "Input recipe".

Units are SI: x [m], G [T/m], B1 [T], dw [rad/s], t [s].
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import dataclasses

import numpy as np

GAMMA = 2.0 * math.pi * 42.58e6  # rad/s/T   (PAPER.md:322 -> 0.267538 rad/us/mT)
GAMMA_BAR = 42.58e6              # Hz/T
SEED0 = 230102702
SLEW = 200.0                     # T/m/s, used for ramp times only
RASTER = 10e-6                   # s, ramp times are multiples of this


@dataclass
class Phantom:
    """Per-spin SoA arrays.  All values are exactly representable in fp32 so that the
    fp32 GPU path and the fp64 oracle see identical inputs."""
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    M0: np.ndarray
    T1: np.ndarray
    T2: np.ndarray
    dw: np.ndarray

    @property
    def n(self) -> int:
        return int(self.x.shape[0])

    def subset(self, idx) -> "Phantom":
        return Phantom(*(np.ascontiguousarray(a[idx]) for a in
                         (self.x, self.y, self.z, self.M0, self.T1, self.T2, self.dw)))


@dataclass
class Sequence:
    """Waveform-level sequence: piecewise-linear gradient vertices per axis (G = 0 outside
    the vertex range), piecewise-constant complex B1 samples, ADC sample times."""
    g_t: list  # 3 arrays of ascending vertex times
    g_v: list  # 3 arrays of vertex values [T/m]
    rf_t: np.ndarray
    rf_dt: np.ndarray
    rf_re: np.ndarray
    rf_im: np.ndarray
    adc_t: np.ndarray
    t_end: float
    dt_rf_max: float = 1e-6
    meta: dict = field(default_factory=dict)


@dataclass
class Workload:
    name: str
    phantom: Phantom
    seq: Sequence
    phase_mode: str = "auto"      # "auto" | "fp32" | "fp64"
    output_mode: str = "sum"      # "sum" | "per_spin"
    velocity: tuple | None = None  # (vx, vy, vz) fp32-exact arrays [m/s]: x(t) = x + v t
    dt_max: float = 0.0            # spacing of the intermediate points needed with motion
    group_size: int = 0            # output_mode "grouped": spins per group
    coils: np.ndarray | None = None  # complex64 [n_coils, n_spins] receive sensitivities (reading C1)
    waveform: tuple | None = None    # (t, u) vertices of a shared motion waveform: x(t) = x + velocity * u(t) (reading M2)

    @property
    def plan_kw(self) -> dict:
        kw = dict(phase_mode=self.phase_mode, output_mode=self.output_mode)
        if self.velocity is not None:
            kw.update(motion="linear", dt_max=self.dt_max)
        if self.waveform is not None:
            kw.update(motion="waveform", waveform=self.waveform)
        if self.output_mode == "grouped":
            kw.update(group_size=self.group_size)
        return kw


def _f32(a):
    return np.asarray(a, dtype=np.float64).astype(np.float32).astype(np.float64)


def _phantom(x, y, z, M0, T1, T2, dw) -> Phantom:
    T1 = np.asarray(T1, dtype=np.float64)
    T2 = np.minimum(np.asarray(T2, dtype=np.float64), 0.95 * T1)   # reading G14
    return Phantom(*(np.ascontiguousarray(_f32(a).ravel()) for a in (x, y, z, M0, T1, T2, dw)))


# --------------------------------------------------------------------------------------------------
# gradient waveform builder: one list of (t, v) vertices per axis
# --------------------------------------------------------------------------------------------------
class _Axis:
    def __init__(self):
        self.t: list[float] = []
        self.v: list[float] = []

    def add(self, t: float, v: float):
        if self.t and t < self.t[-1] - 1e-12:
            raise ValueError(f"gradient vertices not ascending: {t} < {self.t[-1]}")
        if self.t and abs(t - self.t[-1]) <= 1e-12:
            if abs(v - self.v[-1]) > 1e-15:
                raise ValueError("gradient discontinuity at a vertex")
            return
        self.t.append(float(t))
        self.v.append(float(v))

    def trap(self, t0: float, amp: float, ramp: float, flat: float) -> float:
        """Trapezoid starting (at zero) at t0; returns its end time."""
        self.add(t0, 0.0)
        self.add(t0 + ramp, amp)
        if flat > 0:
            self.add(t0 + ramp + flat, amp)
        self.add(t0 + 2 * ramp + flat, 0.0)
        return t0 + 2 * ramp + flat

    def arrays(self):
        return np.asarray(self.t, dtype=np.float64), np.asarray(self.v, dtype=np.float64)


def _ramp_time(amp: float) -> float:
    return max(1, math.ceil(abs(amp) / SLEW / RASTER - 1e-9)) * RASTER


def _area_trap(area_k: float, max_amp: float = 30e-3):
    """Design a trapezoid (amp, ramp, flat) whose k-space area (in 1/m, i.e. gamma_bar * integral G) is
    area_k.  Ramp from the slew limit, flat on the 10 us raster."""
    if area_k == 0.0:
        return 0.0, RASTER, 0.0
    a = abs(area_k) / GAMMA_BAR           # T/m * s
    ramp = _ramp_time(max_amp)
    flat = max(0.0, math.ceil((a / max_amp - ramp) / RASTER - 1e-9) * RASTER)
    amp = a / (ramp + flat)
    return math.copysign(amp, area_k), ramp, flat


def _sinc_rf(t0: float, dur: float, n: int, flip: float, tbw: float = 4.0, phase: float = 0.0):
    """Un-apodised sinc envelope sampled at step midpoints, scaled so gamma*sum(B1*dt) = flip exactly
    (reading G6)."""
    dt = dur / n
    tm = (np.arange(n) + 0.5) * dt
    env = np.sinc(tbw * (tm - dur / 2) / dur)
    b1 = env * (flip / (GAMMA * dt * env.sum()))
    rf_t = t0 + np.arange(n) * dt
    return rf_t, np.full(n, dt), b1 * math.cos(phase), b1 * math.sin(phase)


def _slice_select(gz: _Axis, t_rf0: float, dur: float, tbw: float, thk: float) -> float:
    """Plateau spanning the RF exactly, ramps outside, then a rephaser of -(half plateau + ramp) area.
    Returns the end time of the rephaser."""
    amp = tbw / (dur * GAMMA_BAR * thk)
    ramp = _ramp_time(amp)
    gz.add(t_rf0 - ramp, 0.0)
    gz.add(t_rf0, amp)
    gz.add(t_rf0 + dur, amp)
    gz.add(t_rf0 + dur + ramp, 0.0)
    area_k = -(0.5 * amp * dur + 0.5 * amp * ramp) * GAMMA_BAR
    a, r, f = _area_trap(area_k)
    return gz.trap(t_rf0 + dur + ramp, a, r, f)


def _finish(axes, rf_parts, adc_parts, t_end, dt_rf_max, meta) -> Sequence:
    g = [ax.arrays() for ax in axes]
    if rf_parts:
        rf = [np.concatenate([p[i] for p in rf_parts]) for i in range(4)]
    else:
        rf = [np.zeros(0)] * 4
    adc = np.concatenate(adc_parts) if adc_parts else np.zeros(0)
    return Sequence([a[0] for a in g], [a[1] for a in g], rf[0], rf[1], rf[2], rf[3],
                    np.ascontiguousarray(adc, dtype=np.float64), float(t_end), dt_rf_max, meta)


def _epi(axes, t0: float, n: int, fov: float, dwell: float):
    """Single-shot Cartesian EPI n x n starting at t0: prephasers to (-n/2 dk, -n/2 dk), alternating
    readout trapezoids, triangular y blips of area dk during the readout ramps.  Returns (adc, t_end)."""
    gx, gy, _ = axes
    dk = 1.0 / fov
    g_read = dk / (GAMMA_BAR * dwell)
    ramp = _ramp_time(g_read)
    flat = n * dwell
    ramp_k = 0.5 * g_read * ramp * GAMMA_BAR
    # prephasers
    ax_, rx_, fx_ = _area_trap(-(n / 2) * dk - ramp_k)
    ay_, ry_, fy_ = _area_trap(-(n / 2) * dk)
    t1 = gx.trap(t0, ax_, rx_, fx_)
    t2 = gy.trap(t0, ay_, ry_, fy_)
    t = max(t1, t2)
    adc = []
    blip_amp = dk / (GAMMA_BAR * ramp)   # triangle of base 2*ramp
    for line in range(n):
        sgn = 1.0 if line % 2 == 0 else -1.0
        gx.add(t, 0.0)
        gx.add(t + ramp, sgn * g_read)
        gx.add(t + ramp + flat, sgn * g_read)
        gx.add(t + 2 * ramp + flat, 0.0)
        adc.append(t + ramp + (np.arange(n) + 0.5) * dwell)
        t_line_end = t + 2 * ramp + flat
        if line < n - 1:
            gy.add(t_line_end - ramp, 0.0)
            gy.add(t_line_end, blip_amp)
            gy.add(t_line_end + ramp, 0.0)
        t = t_line_end
    return np.concatenate(adc), t


# --------------------------------------------------------------------------------------------------
# phantoms
# --------------------------------------------------------------------------------------------------
def _grid(n: int, fov: float):
    return ((np.arange(n) + 0.5) / n - 0.5) * fov


def _classes3(x, y, rng, scale=1.0):
    rho = np.sqrt((x / (0.09 * scale)) ** 2 + (y / (0.075 * scale)) ** 2)
    T1 = np.where(rho < 0.35, 4.0, np.where(rho < 0.7, 0.8, 1.3))
    T2 = np.where(rho < 0.35, 2.0, np.where(rho < 0.7, 0.07, 0.11))
    M0 = np.where(rho < 0.35, 1.0, np.where(rho < 0.7, 0.7, 0.8))
    n = x.shape[0]
    M0 = M0 * (1 + rng.uniform(-0.05, 0.05, n))
    T1 = T1 * (1 + rng.uniform(-0.05, 0.05, n))
    T2 = T2 * (1 + rng.uniform(-0.05, 0.05, n))
    return M0, T1, T2


# --------------------------------------------------------------------------------------------------
# config 1: tiny 2-D, hard pulse + EPI 32x32
# --------------------------------------------------------------------------------------------------
def config1(n_grid: int = 32, n_epi: int = 32) -> Workload:
    rng = np.random.default_rng(SEED0 + 1)
    fov = 0.2
    g = _grid(n_grid, fov)
    X, Y = np.meshgrid(g, g, indexing="ij")
    n = n_grid * n_grid
    M0 = rng.uniform(0, 1, n)
    T1 = rng.uniform(0.3, 2.0, n)
    T2 = rng.uniform(0.03, 0.3, n)
    ph = _phantom(X.ravel(), Y.ravel(), np.zeros(n), M0, T1, T2, np.zeros(n))

    axes = [_Axis(), _Axis(), _Axis()]
    dur, nrf = 0.5e-3, 50
    dt = dur / nrf
    b1 = (math.pi / 2) / (GAMMA * dur)
    rf = (np.arange(nrf) * dt, np.full(nrf, dt), np.full(nrf, b1), np.zeros(nrf))
    adc, t = _epi(axes, dur + 20e-6, n_epi, fov, 10e-6)
    t_end = t + 100e-6
    seq = _finish(axes, [rf], [adc], t_end, 10e-6, {"config": 1})
    return Workload("config1_tiny_epi32", ph, seq)


# --------------------------------------------------------------------------------------------------
# config 2: GRE 64x64 on a 64x64x4 grid
# --------------------------------------------------------------------------------------------------
def config2(n_grid: int = 64, n_pe: int = 64, n_ro: int = 64, n_rf: int = 1000) -> Workload:
    rng = np.random.default_rng(SEED0 + 2)
    fov = 0.2
    g = _grid(n_grid, fov)
    zs = (np.arange(4) - 1.5) * 1.25e-3
    X, Y, Z = np.meshgrid(g, g, zs, indexing="ij")
    x, y, z = X.ravel(), Y.ravel(), Z.ravel()
    M0, T1, T2 = _classes3(x, y, rng)
    ph = _phantom(x, y, z, M0, T1, T2, np.zeros_like(x))

    TR, TE, dur, dwell, thk = 20e-3, 5e-3, 1e-3, 8e-6, 5e-3
    dk = 1.0 / fov
    g_read = dk / (GAMMA_BAR * dwell)
    ramp = _ramp_time(g_read)
    flat = n_ro * dwell
    axes = [_Axis(), _Axis(), _Axis()]
    rf_parts, adc_parts = [], []
    t_lead = 200e-6
    for k in range(n_pe):
        t0 = k * TR + t_lead
        rf_parts.append(_sinc_rf(t0, dur, n_rf, math.radians(15.0)))
        t_reph = _slice_select(axes[2], t0, dur, 4.0, thk)
        # readout centred at TE from RF centre
        t_ro0 = t0 + dur / 2 + TE - flat / 2 - ramp
        ramp_k = 0.5 * g_read * ramp * GAMMA_BAR
        ax_, rx_, fx_ = _area_trap(-(n_ro / 2) * dk - ramp_k)
        ell = k - n_pe // 2
        ay_, ry_, fy_ = _area_trap(ell * dk)
        t_pre = max(t_reph, t0 + dur) + 10e-6
        axes[0].trap(t_pre, ax_, rx_, fx_)
        if ell != 0:
            axes[1].trap(t_pre, ay_, ry_, fy_)
        axes[0].trap(t_ro0, g_read, ramp, flat)
        adc_parts.append(t_ro0 + ramp + (np.arange(n_ro) + 0.5) * dwell)
    seq = _finish(axes, rf_parts, adc_parts, n_pe * TR, dur / n_rf, {"config": 2})
    return Workload("config2_gre64", ph, seq)


# --------------------------------------------------------------------------------------------------
# config 3: brain-like slice, slice-selective 90 + EPI 128x128, fp64 phase
# --------------------------------------------------------------------------------------------------
def config3(n_grid: int = 256, n_epi: int = 128, n_rf: int = 1000) -> Workload:
    rng = np.random.default_rng(SEED0 + 3)
    fov = 0.2
    g = _grid(n_grid, fov)
    zs = np.array([-1.25e-3, 1.25e-3])
    X, Y, Z = np.meshgrid(g, g, zs, indexing="ij")
    x, y, z = X.ravel(), Y.ravel(), Z.ravel()
    cls = np.zeros(x.shape[0], dtype=np.int64)
    for c in range(1, 6):
        cx, cy = rng.uniform(-0.06, 0.06, 2)
        a, b = rng.uniform(0.01, 0.05, 2)
        th = rng.uniform(0, math.pi)
        u = (x - cx) * math.cos(th) + (y - cy) * math.sin(th)
        v = -(x - cx) * math.sin(th) + (y - cy) * math.cos(th)
        cls[(u / a) ** 2 + (v / b) ** 2 < 1.0] = c
    T1c = rng.uniform(0.4, 4.0, 6)
    T2c = rng.uniform(0.04, 2.0, 6)
    M0c = rng.uniform(0.5, 1.0, 6)
    coef = rng.uniform(-1, 1, 6)
    u, v = x / (fov / 2), y / (fov / 2)
    df = coef[0] + coef[1] * u + coef[2] * v + coef[3] * u * u + coef[4] * u * v + coef[5] * v * v
    df = df * (100.0 / np.abs(df).max())
    ph = _phantom(x, y, z, M0c[cls], T1c[cls], T2c[cls], 2 * math.pi * df)

    axes = [_Axis(), _Axis(), _Axis()]
    dur, thk = 1e-3, 5e-3
    t0 = 200e-6
    rf = _sinc_rf(t0, dur, n_rf, math.pi / 2)
    t_reph = _slice_select(axes[2], t0, dur, 4.0, thk)
    adc, t = _epi(axes, t_reph + 10e-6, n_epi, fov, 4e-6)
    seq = _finish(axes, [rf], [adc], t + 100e-6, dur / n_rf, {"config": 3})
    return Workload("config3_brain_epi128", ph, seq, phase_mode="fp64")


# --------------------------------------------------------------------------------------------------
# spiral helper (configs 4, 5)
# --------------------------------------------------------------------------------------------------
def _spiral(axes, t0: float, n_samp: int, dwell: float, k_max: float, turns: float, rot: float):
    """Variable-density spiral k(s) = k_max s^2 exp(i(2 pi N s + rot)), s = t/T_read.  Gradient vertices
    at every dwell boundary hold the analytic dk/dt / gamma_bar; then a linear ramp to zero and one
    rewinder trapezoid per axis that returns k to 0.  Returns (adc_times, t_end)."""
    T = n_samp * dwell
    s = np.arange(n_samp + 1) / n_samp
    ang = 2 * math.pi * turns * s + rot
    dk_ds = k_max * (2 * s + 1j * 2 * math.pi * turns * s * s) * np.exp(1j * ang)
    G = dk_ds / T / GAMMA_BAR
    tv = t0 + np.arange(n_samp + 1) * dwell
    t_ends = []
    for ax, Gv in ((axes[0], G.real), (axes[1], G.imag)):
        for ti, vi in zip(tv, Gv):
            ax.add(float(ti), float(vi))
        # trapezoid-rule moment of the sampled waveform, as both solvers integrate it
        k_end = GAMMA_BAR * float(np.sum(0.5 * (Gv[1:] + Gv[:-1]) * dwell))
        ramp = _ramp_time(Gv[-1]) if Gv[-1] != 0.0 else RASTER
        t_r = float(tv[-1]) + ramp
        ax.add(t_r, 0.0)
        k_end += GAMMA_BAR * 0.5 * float(Gv[-1]) * ramp
        a, r, f = _area_trap(-k_end)
        t_ends.append(ax.trap(t_r, a, r, f))
    adc = t0 + (np.arange(n_samp) + 0.5) * dwell
    return adc, max(t_ends)


# --------------------------------------------------------------------------------------------------
# config 4: 1M-spin slab, 16-interleave spiral
# --------------------------------------------------------------------------------------------------
def config4(n_spins: int = 1_000_000, n_shots: int = 16, n_samp: int = 4096, n_rf: int = 2000,
            turns: float = 8.0) -> Workload:
    rng = np.random.default_rng(SEED0 + 4)
    x = rng.uniform(-0.11, 0.11, n_spins)
    y = rng.uniform(-0.11, 0.11, n_spins)
    z = rng.uniform(-0.01, 0.01, n_spins)
    M0, T1, T2 = _classes3(x, y, rng, scale=1.1)
    df = rng.uniform(-50.0, 50.0, n_spins)
    ph = _phantom(x, y, z, M0, T1, T2, 2 * math.pi * df)

    TR, dur, thk, dwell = 15e-3, 2e-3, 20e-3, 2e-6
    k_max = 128 / (2 * 0.22)
    axes = [_Axis(), _Axis(), _Axis()]
    rf_parts, adc_parts = [], []
    for j in range(n_shots):
        t0 = j * TR + 200e-6
        rf_parts.append(_sinc_rf(t0, dur, n_rf, math.radians(30.0)))
        t_reph = _slice_select(axes[2], t0, dur, 4.0, thk)
        adc, _ = _spiral(axes, t_reph + 10e-6, n_samp, dwell, k_max, turns, 2 * math.pi * j / n_shots)
        adc_parts.append(adc)
    seq = _finish(axes, rf_parts, adc_parts, n_shots * TR, dur / n_rf, {"config": 4})
    return Workload("config4_1M_spiral", ph, seq)


# --------------------------------------------------------------------------------------------------
# config 5 / 5b: MRF FISP
# --------------------------------------------------------------------------------------------------
def _mrf_sequence(n_tr: int, n_samp: int, n_rf: int, one_adc_per_tr: bool, rng, turns: float = 6.0) -> Sequence:
    k = np.arange(n_tr)
    fa = np.clip(37.5 + 32.5 * np.sin(2 * math.pi * k / 250.0) + 2.0 * rng.standard_normal(n_tr), 5.0, 70.0)
    TRs = rng.uniform(10e-3, 15e-3, n_tr)
    TRs = np.round(TRs / 1e-6) * 1e-6            # on a 1 us raster
    dur, dwell = 1e-3, 2e-6
    golden = math.pi * (3.0 - math.sqrt(5.0))
    axes = [_Axis(), _Axis(), _Axis()]
    rf_parts, adc_parts = [], []
    t_tr = 0.0
    for i in range(n_tr):
        t0 = t_tr + 100e-6
        rf_parts.append(_sinc_rf(t0, dur, n_rf, math.radians(float(fa[i]))))
        adc, t_sp = _spiral(axes, t0 + dur + 500e-6, n_samp, dwell, 128.0, turns, golden * i)
        adc_parts.append(adc[:1] if one_adc_per_tr else adc)
        a, r, f = _area_trap(320.0)              # x-axis spoiler, 320 1/m
        axes[0].trap(t_sp + 10e-6, a, r, f)
        t_tr += float(TRs[i])
    return _finish(axes, rf_parts, adc_parts, t_tr, dur / n_rf,
                   {"config": 5, "fa_deg": fa, "TR": TRs})


def config5(n_grid: int = 256, n_tr: int = 1000, n_samp: int = 1024, n_rf: int = 1000,
            turns: float = 6.0) -> Workload:
    rng = np.random.default_rng(SEED0 + 5)
    fov = 0.2
    g = _grid(n_grid, fov)
    X, Y = np.meshgrid(g, g, indexing="ij")
    n = n_grid * n_grid
    T1 = rng.uniform(0.1, 4.0, n)
    T2 = rng.uniform(0.01, 0.6, n)
    ph = _phantom(X.ravel(), Y.ravel(), np.zeros(n), np.ones(n), T1, T2, np.zeros(n))
    seq = _mrf_sequence(n_tr, n_samp, n_rf, False, rng, turns)
    return Workload("config5_mrf_fisp", ph, seq)


def config5b(n_entries: int = 100_000, n_tr: int = 1000, n_samp: int = 1024, n_rf: int = 1000,
             turns: float = 6.0) -> Workload:
    """Dictionary mode: the phantom draws come from their own stream; the schedule is config 5's
    (same seed, same draw order for the sequence part)."""
    rng5 = np.random.default_rng(SEED0 + 5)
    n5 = 256 * 256
    rng5.uniform(0.1, 4.0, n5)
    rng5.uniform(0.01, 0.6, n5)                  # skip config 5's phantom draws -> same schedule
    seq = _mrf_sequence(n_tr, n_samp, n_rf, True, rng5, turns)
    rng = np.random.default_rng(SEED0 + 6)
    T1 = rng.uniform(0.1, 4.0, n_entries)
    T2 = rng.uniform(0.01, 0.6, n_entries)
    z = np.zeros(n_entries)
    ph = _phantom(z, z, z, np.ones(n_entries), T1, T2, z)
    return Workload("config5b_mrf_dictionary", ph, seq, output_mode="per_spin")


def config5c(n_entries: int = 10_000, n_iso: int = 64, n_tr: int = 1000, n_samp: int = 1024, n_rf: int = 1000,
             turns: float = 6.0) -> Workload:
    """Ensemble dictionary: config 5b's schedule, but every (T1, T2) entry is n_iso
    isochromats spread evenly over one period of the x spoiler (320 1/m -> 3.125 mm), so that an entry's
    GROUPED signal is a proper FISP ensemble (PAPER.md:167 "use more spins", :368).  Output
    [entry][TR] complex."""
    w = config5b(n_entries, n_tr, n_samp, n_rf, turns)
    period = 1.0 / 320.0
    xk = ((np.arange(n_iso) + 0.5) / n_iso - 0.5) * period
    T1 = np.repeat(w.phantom.T1, n_iso)
    T2 = np.repeat(w.phantom.T2, n_iso)
    n = n_entries * n_iso
    z = np.zeros(n)
    ph = _phantom(np.tile(xk, n_entries), z, z, np.full(n, 1.0 / n_iso), T1, T2, z)
    return Workload("config5c_mrf_ensemble_dictionary", ph, w.seq, output_mode="grouped", group_size=n_iso)


def config3m(n_grid: int = 256, n_epi: int = 128, n_rf: int = 1000, vy: float = 0.1, dt_max: float = 1e-5) -> Workload:
    """Config 3 without off-resonance but with motion, the paper's experiment (d):
    u_y(x, t) = v_y t with v_y = 0.1 m/s for every spin; intermediate points every dt_max."""
    w = config3(n_grid, n_epi, n_rf)
    ph = w.phantom
    n = ph.n
    ph = Phantom(ph.x, ph.y, ph.z, ph.M0, ph.T1, ph.T2, np.zeros(n))
    vel = (np.zeros(n), _f32(np.full(n, vy)), np.zeros(n))
    return Workload("config3m_brain_epi128_motion", ph, w.seq, phase_mode="fp64", velocity=vel, dt_max=dt_max)


def config3w(n_grid: int = 256, n_epi: int = 128, n_rf: int = 1000, dt_max: float = 1e-5) -> Workload:
    """Config 3 (off-resonance included) under NON-RIGID periodic motion, the general motion field u(x, t) of
    PAPER.md:96 in its separable form x(t) = x + a(x) u(t): u(t) = sin(2 pi t / 50 ms) given by 101 vertices per period
    (a breathing-like displacement, sped up so that the 73 ms EPI sees one and a half periods), amplitude growing
    from 0.5 mm to 2.5 mm along y (in-plane stretch) plus a 0.3 mm through-slice part; intermediate points every dt_max."""
    w = config3(n_grid, n_epi, n_rf)
    ph = w.phantom
    period = 50e-3
    n_v = int(math.ceil(w.seq.t_end / period * 100)) + 1
    wt = np.arange(n_v) * (period / 100)
    wu = np.sin(2 * math.pi * wt / period)
    ay = 1.5e-3 + 1e-3 * (ph.y / 0.1)
    amp = (np.zeros(ph.n), _f32(ay), _f32(np.full(ph.n, 0.3e-3)))
    return Workload("config3w_brain_epi128_periodic_motion", ph, w.seq, phase_mode="fp64", velocity=amp, dt_max=dt_max,
                    waveform=(wt, wu))


def coil_maps(ph: Phantom, n_coils: int, radius: float = 0.15, seed: int = 0) -> np.ndarray:
    """Smooth synthetic receive sensitivities, complex64 [n_coils, n_spins]: coils on a ring of `radius` around the
    z axis, magnitude r0^2 / (d^2 + r0^2) with d the in-plane distance to the coil and r0 = 0.1 m, phase = the angle
    from the coil to the spin (a Biot-Savart-like stand-in for measured maps, which are not in this container)."""
    rng = np.random.default_rng(SEED0 + 40 + seed)
    ang = 2 * np.pi * (np.arange(n_coils) + rng.uniform(0, 1)) / n_coils
    cx, cy = radius * np.cos(ang), radius * np.sin(ang)
    dx, dy = ph.x[None, :] - cx[:, None], ph.y[None, :] - cy[:, None]
    w = 0.01 / (dx * dx + dy * dy + 0.01) * np.exp(1j * np.arctan2(dy, dx))
    return w.astype(np.complex64)


def config4c(n_coils: int = 8, **kw) -> Workload:
    """Config 4 received by 8 coils (SURVEY.md 8(f) f2 "per-coil weights"): output 8 x 65,536 complex."""
    w = config4(**kw)
    return dataclasses.replace(w, name=f"config4c_1M_spiral_{n_coils}coils", coils=coil_maps(w.phantom, n_coils))


def with_coils(base: str, n_coils: int, **kw) -> Workload:
    """Config `base` received by n_coils synthetic coils ("5x8": config 5 with 8 coils -- the multi-coil sums inside
    the whole-sequence kernel, f2 x a5-a8)."""
    w = CONFIGS[base](**kw)
    return dataclasses.replace(w, name=f"{w.name}_x{n_coils}coils", coils=coil_maps(w.phantom, n_coils))


CONFIGS = {"1": config1, "2": config2, "3": config3, "3m": config3m, "3w": config3w, "4": config4, "5": config5, "5b": config5b,
           "5c": config5c, "4c": config4c,
           "4c32": lambda **kw: config4c(n_coils=32, **kw)}


def make(name: str, **kw) -> Workload:
    name = str(name)
    if name not in CONFIGS and "x" in name:   # "<config>x<n_coils>", e.g. "5x8", "2x4"
        base, n_coils = name.split("x")
        return with_coils(base, int(n_coils), **kw)
    return CONFIGS[name](**kw)


def small(name: str) -> Workload:
    """Reduced-size variants (same structure) that the CPU oracle finishes in seconds; used by the
    parity tests.  Sizes still span several kernel tiles and leave ragged tails.  Spiral turn counts are
    scaled with the shortened readouts so that the gradient amplitudes stay those of the full configs."""
    name = str(name)
    if name == "1":
        return config1()
    if name == "2":
        return config2(n_grid=24, n_pe=6, n_ro=64, n_rf=200)
    if name == "3":
        return config3(n_grid=48, n_epi=32, n_rf=250)
    if name == "3m":
        return config3m(n_grid=24, n_epi=16, n_rf=100)
    if name == "3w":
        return config3w(n_grid=24, n_epi=16, n_rf=100)
    if name == "4":
        return config4(n_spins=5003, n_shots=3, n_samp=700, n_rf=300, turns=8.0 * 700 / 4096)
    if name == "5":
        return config5(n_grid=40, n_tr=12, n_samp=300, n_rf=200, turns=6.0 * 300 / 1024)
    if name == "5b":
        return config5b(n_entries=777, n_tr=40, n_samp=512, n_rf=200, turns=3.0)
    if name == "5c":
        return config5c(n_entries=41, n_iso=24, n_tr=40, n_samp=512, n_rf=200, turns=3.0)
    raise KeyError(name)
