"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-type the oracle's formulas: they use closed forms (free precession, hard-pulse flips,
steady states, Dirichlet kernel), scipy's matrix exponential of the Eq (3) generator, linear-algebra fixed
points and invariants.  The paper prints no signal values for this path, so there is no golden number from
the paper itself ("parity unpinned" against the paper's own numbers).
"""
import math

import numpy as np
import pytest
from scipy.linalg import expm

from seqtools import phantom, seq

GAMMA = 2.0 * math.pi * 42.58e6


# ---------------------------------------------------------------------------------------------- P1
def test_p1_free_relaxation_precession_closed_form(oracle_mod):
    T1, T2, dw, M0 = 0.8, 0.07, 2 * math.pi * 37.0, 0.9
    ph = phantom(M0=M0, T1=T1, T2=T2, dw=dw)
    adc = np.array([0.0, 1e-3, 7.3e-3, 20e-3, 50e-3])
    s = seq(adc=adc, t_end=60e-3)
    mxy0 = 1j * M0
    sig, mxy, mz = oracle_mod.simulate(ph, s, state=(np.array([mxy0]), np.array([0.0])), return_state=True)
    want = mxy0 * np.exp(-adc / T2) * np.exp(-1j * dw * adc)      # BASELINE.json north_star closed form
    np.testing.assert_allclose(sig, want, rtol=0, atol=1e-12)
    assert abs(mz[0] - M0 * (1 - math.exp(-60e-3 / T1))) < 1e-12
    # any step partition gives the same value: add zero-valued gradient vertices to force extra points
    tt = np.linspace(0, 60e-3, 977)
    s2 = seq(g={0: (tt, np.zeros_like(tt))}, adc=adc, t_end=60e-3)
    sig2 = oracle_mod.simulate(ph, s2, state=(np.array([mxy0]), np.array([0.0])))
    np.testing.assert_allclose(sig2, want, rtol=0, atol=1e-12)


# ---------------------------------------------------------------------------------------------- P2
def test_p2_gradient_phase_is_minus_gamma_x_area(oracle_mod):
    x = np.array([0.013, -0.05, 0.1])
    ph = phantom(x=x, y=0.02, z=-0.01)
    G = 7e-3
    # trapezoid on x with only 4 vertices; constant y gradient via plateau with ramps
    gx = (np.array([1e-3, 1.2e-3, 2.2e-3, 2.4e-3]), np.array([0.0, G, G, 0.0]))
    gy = (np.array([0.5e-3, 0.6e-3, 2.9e-3, 3.0e-3]), np.array([0.0, -3e-3, -3e-3, 0.0]))
    adc = np.array([0.9e-3, 1.1e-3, 1.7e-3, 2.3e-3, 3.5e-3])
    s = seq(g={0: gx, 1: gy}, adc=adc, t_end=4e-3)
    st = (np.full(3, 1.0 + 0j), np.zeros(3))
    sig = oracle_mod.simulate(ph, s, output_mode="per_spin", state=st)

    def area(tv, t):  # exact integral of the piecewise-linear waveform up to t
        ts, vs = tv
        tt = np.union1d(ts[ts < t], [t])
        vv = np.interp(tt, ts, vs, left=0.0, right=0.0)
        return np.trapezoid(vv, tt) if len(tt) > 1 else 0.0

    for j, t in enumerate(adc):
        ph_want = -GAMMA * (x * area(gx, t) + 0.02 * area(gy, t))
        np.testing.assert_allclose(sig[:, j], np.exp(1j * ph_want), rtol=0, atol=2e-10)
    # full lobe: phase = -gamma x * area of the trapezoid
    full = -GAMMA * (x * G * 1.2e-3 + 0.02 * (-3e-3) * 2.4e-3)
    np.testing.assert_allclose(sig[:, -1], np.exp(1j * full), rtol=0, atol=2e-10)


# ---------------------------------------------------------------------------------------------- P3
@pytest.mark.parametrize("theta_deg", [90.0, 30.0, 180.0, 7.0])
def test_p3_hard_pulse_flip_angle_and_axis(oracle_mod, theta_deg):
    th = math.radians(theta_deg)
    T = 0.4e-3
    b1 = th / (GAMMA * T)
    ph = phantom(M0=0.8)
    for arg, want in ((0.0, (0.0, math.sin(th), math.cos(th))),            # +x B1 tips +z toward +y (G3)
                      (math.pi / 2, (-math.sin(th), 0.0, math.cos(th)))):  # +y B1 tips toward -x
        for dt_rf in (T, T / 7, 1e-6):                                      # independent of sub-stepping
            s = seq(rf=([0.0], [T], [b1 * math.cos(arg)], [b1 * math.sin(arg)]), t_end=T, dt_rf_max=dt_rf)
            _, mxy, mz = oracle_mod.simulate(ph, s, return_state=True)
            got = np.array([mxy[0].real, mxy[0].imag, mz[0]]) / 0.8
            np.testing.assert_allclose(got, want, rtol=0, atol=1e-12)


# ---------------------------------------------------------------------------------------------- P4
def _omega(bx, by, bz):
    """Generator of Eq (3)."""
    return GAMMA * np.array([[0, bz, -by], [-bz, 0, bx], [by, -bx, 0]])


def test_p4_offresonant_hard_pulse_matches_expm_and_rodrigues(oracle_mod):
    rng = np.random.default_rng(4)
    for _ in range(20):
        b1x, b1y = rng.normal(0, 8e-6, 2)
        dw = rng.normal(0, 2e4)
        T = rng.uniform(0.1e-3, 1e-3)
        m0 = rng.normal(0, 1, 3)
        ph = phantom(M0=1.0, dw=dw)
        s = seq(rf=([0.0], [T], [b1x], [b1y]), t_end=T, dt_rf_max=T)
        _, mxy, mz = oracle_mod.simulate(ph, s, state=(np.array([m0[0] + 1j * m0[1]]), np.array([m0[2]])),
                                         return_state=True)
        got = np.array([mxy[0].real, mxy[0].imag, mz[0]])
        bz = dw / GAMMA
        want = expm(_omega(b1x, b1y, bz) * T) @ m0
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-11)
        # Rodrigues: dM/dt = gamma M x B is a LEFT-handed rotation about B by gamma|B|T
        B = np.array([b1x, b1y, bz])
        nB = np.linalg.norm(B)
        n = B / nB
        ang = -GAMMA * nB * T
        rod = m0 * math.cos(ang) + np.cross(n, m0) * math.sin(ang) + n * (n @ m0) * (1 - math.cos(ang))
        np.testing.assert_allclose(got, rod, rtol=0, atol=1e-11)


# ---------------------------------------------------------------------------------------------- P5
def test_p5_bruteforce_matrix_products(oracle_mod):
    """Whole RF path incl. the Eq (11) interleaving: product over steps of expm(Omega dt) then relaxation."""
    rng = np.random.default_rng(5)
    n_sp, n_st = 6, 48
    dt = 10e-6
    x = rng.uniform(-0.1, 0.1, n_sp); y = rng.uniform(-0.1, 0.1, n_sp); z = rng.uniform(-0.01, 0.01, n_sp)
    M0 = rng.uniform(0.5, 1, n_sp); T1 = rng.uniform(0.002, 0.01, n_sp); T2 = rng.uniform(0.0005, 0.002, n_sp)
    dw = rng.normal(0, 3e3, n_sp)
    ph = phantom(x, y, z, M0, T1, T2, dw)
    rf_t = np.arange(n_st) * dt
    b1 = rng.normal(0, 30e-6, n_st) + 1j * rng.normal(0, 30e-6, n_st)
    tv = np.arange(n_st + 1) * dt                     # gradient vertices on the RF edges, piecewise linear
    gv = [rng.normal(0, 5e-3, n_st + 1) for _ in range(3)]
    for a in range(3):
        gv[a][0] = 0.0
        gv[a][-1] = 0.0
    adc = tv[[5, 17, n_st]]
    s = seq(g={a: (tv, gv[a]) for a in range(3)}, rf=(rf_t, np.full(n_st, dt), b1.real, b1.imag),
            adc=adc, t_end=n_st * dt, dt_rf_max=dt)
    sig, mxy, mz = oracle_mod.simulate(ph, s, output_mode="per_spin", return_state=True)
    for i in range(n_sp):
        M = np.array([0.0, 0.0, M0[i]])
        rec = {}
        for n in range(n_st):
            gbar = [0.5 * (gv[a][n] + gv[a][n + 1]) for a in range(3)]   # reading G5
            bz = gbar[0] * x[i] + gbar[1] * y[i] + gbar[2] * z[i] + dw[i] / GAMMA
            M = expm(_omega(b1[n].real, b1[n].imag, bz) * dt) @ M
            E1, E2 = math.exp(-dt / T1[i]), math.exp(-dt / T2[i])
            M = np.array([E2 * M[0], E2 * M[1], E1 * M[2] + M0[i] * (1 - E1)])
            rec[n + 1] = M.copy()
        for j, n in enumerate((5, 17, n_st)):
            assert abs(sig[i, j] - (rec[n][0] + 1j * rec[n][1])) < 1e-11
        assert abs(mz[i] - M[2]) < 1e-11 and abs(mxy[i] - (M[0] + 1j * M[1])) < 1e-11


# ---------------------------------------------------------------------------------------------- P6
def test_p6_spin_echo_refocuses_offresonance_and_gradient(oracle_mod):
    tp = 1e-9                                     # near-instantaneous pulses
    tau = 8e-3
    T2 = 0.06
    dw = np.array([0.0, 150.0, -600.0, 2500.0])
    x = np.array([0.0, 0.03, -0.08, 0.1])
    ph = phantom(x=x, M0=1.0, T1=1e30, T2=T2, dw=dw)
    b90 = (math.pi / 2) / (GAMMA * tp)
    b180 = math.pi / (GAMMA * tp)
    t180 = tp + tau
    # constant x gradient during both free periods (ramps of 1 us, same area each side)
    G = 2e-3
    g = (np.array([10e-6, 11e-6, tau - 100e-6, tau - 99e-6, t180 + tp + 10e-6, t180 + tp + 11e-6,
                   t180 + tp + tau - 100e-6, t180 + tp + tau - 99e-6]),
         np.array([0, G, G, 0, 0, G, G, 0.0]))
    t_echo = t180 + tp + tau
    s = seq(g={0: g}, rf=([0.0, t180], [tp, tp], [b90, 0.0], [0.0, b180]), adc=[t_echo], t_end=t_echo,
            dt_rf_max=tp)
    sig = oracle_mod.simulate(ph, s, output_mode="per_spin")[:, 0]
    # 90x gives Mxy = +i; 180y maps Mxy -> -conj(Mxy) = +i ... the echo re-forms along the same axis
    want = 1j * math.exp(-(2 * tau + 2 * tp) / T2)
    # tolerance O(dw * tp) and gradient*tp
    np.testing.assert_allclose(sig, np.full(4, want), rtol=0, atol=2e-5)


# ---------------------------------------------------------------------------------------------- P7
def _periodic(oracle_mod, alpha, TR, T1, T2, n_tr, dws, alternate, adc_after, adc_before):
    tp = 1e-9
    b = alpha / (GAMMA * tp)
    rf_t = np.arange(n_tr) * TR
    sign = np.where(np.arange(n_tr) % 2 == 0, 1.0, -1.0) if alternate else np.ones(n_tr)
    adc = []
    if adc_after:
        adc.append(rf_t[-1] + tp)
    if adc_before:
        adc.append(rf_t[-1])
    adc = np.sort(np.array(adc))
    s = seq(rf=(rf_t, np.full(n_tr, tp), b * sign, np.zeros(n_tr)), adc=adc, t_end=rf_t[-1] + TR, dt_rf_max=tp)
    ph = phantom(M0=1.0, T1=T1, T2=T2, dw=dws)
    return oracle_mod.simulate(ph, s, output_mode="per_spin")


def test_p7_bssfp_steady_state(oracle_mod):
    alpha, TR, T1, T2 = math.radians(40.0), 5e-3, 0.12, 0.05
    E1, E2 = math.exp(-TR / T1), math.exp(-TR / T2)
    sig = _periodic(oracle_mod, alpha, TR, T1, T2, 400, 0.0, True, True, False)
    want = (1 - E1) * math.sin(alpha) / (1 - (E1 - E2) * math.cos(alpha) - E1 * E2)
    assert abs(abs(sig[0, 0]) - want) < 1e-7


def test_p7_fisp_fid_and_echo_steady_state(oracle_mod):
    alpha, TR, T1, T2 = math.radians(25.0), 6e-3, 0.1, 0.04
    E1, E2 = math.exp(-TR / T1), math.exp(-TR / T2)
    n_iso = 256
    dws = 2 * math.pi * np.arange(n_iso) / (n_iso * TR)   # spoiler phase uniformly covering 2 pi per TR
    sig = _periodic(oracle_mod, alpha, TR, T1, T2, 300, dws, False, True, True)
    m_before, m_after = sig[:, 0].mean(), sig[:, 1].mean()
    ca = math.cos(alpha)
    r = math.sqrt((1 - E2 ** 2) / ((1 - E1 * ca) ** 2 - E2 ** 2 * (E1 - ca) ** 2))
    fid = math.tan(alpha / 2) * (1 - (E1 - ca) * r)
    echo = math.tan(alpha / 2) * (1 - (1 - E1 * ca) * r)
    assert abs(abs(m_after) - fid) < 1e-6
    assert abs(abs(m_before) - abs(echo)) < 1e-6


def test_p7_fixed_point_linear_algebra(oracle_mod):
    """Arbiter: steady state M = (I - A)^-1 b of one TR built from Eq (3)/(4) operators."""
    alpha, TR, T1, T2, dw = math.radians(33.0), 7e-3, 0.09, 0.03, 211.0
    tp = 1e-9
    sig = _periodic(oracle_mod, alpha, TR, T1, T2, 300, dw, False, True, False)
    R = expm(_omega(alpha / (GAMMA * tp), 0.0, dw / GAMMA) * tp)
    P = expm(_omega(0.0, 0.0, dw / GAMMA) * (TR - tp))
    E = np.diag([math.exp(-(TR - tp) / T2)] * 2 + [math.exp(-(TR - tp) / T1)])
    bvec = np.array([0, 0, 1 - math.exp(-(TR - tp) / T1)])
    # M_after = R (E P M_after + b)
    A = R @ E @ P
    M = np.linalg.solve(np.eye(3) - A, R @ bvec)
    assert abs(sig[0, 0] - (M[0] + 1j * M[1])) < 1e-7


# ---------------------------------------------------------------------------------------------- P8
def test_p8_dirichlet_kernel_and_echo_centre(oracle_mod):
    N, dx = 16, 0.0125
    xs = (np.arange(N) - (N - 1) / 2) * dx
    ph = phantom(x=xs)
    G, Tg = 1e-3, 4e-3
    tv = np.array([0.0, 1e-6, Tg, Tg + 1e-6])
    adc = np.linspace(10e-6, Tg - 10e-6, 41)
    s = seq(g={0: (tv, np.array([0, G, G, 0.0]))}, adc=adc, t_end=Tg + 2e-6)
    sig = oracle_mod.simulate(ph, s, state=(np.ones(N, dtype=complex), np.zeros(N)))
    k = (GAMMA / (2 * math.pi)) * G * (adc - 0.5e-6)          # cycles / m
    want = np.sin(math.pi * k * N * dx) / np.sin(math.pi * k * dx)   # centred grid -> real kernel
    np.testing.assert_allclose(sig, want, rtol=0, atol=1e-9)


def test_p8_paper_phantoms_echo_centre_sum(oracle_mod):
    """Phantoms (a) and (b) of PAPER.md:232-233 (geometry in tests/golden/paper_phantoms.txt): at k = 0,
    after an instantaneous +x pulse of angle theta, S = i sin(theta) sum M0 exp(-TE/T2) exp(-i dw TE)."""
    import os
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_phantoms.txt")) as f:
        for line in f:
            if line.startswith("#") or "=" not in line:
                continue
            k, v = line.split("=", 1)
            vals[k.strip()] = [float(u) for u in v.split(",")]
    # (a) column of four 50 mm segments, 1 mm spacing
    ys = (np.arange(200) + 0.5) * 1e-3 - 0.1
    seg = np.minimum((ys + 0.1) // 0.05, 3).astype(int)
    M0 = np.array(vals["a_M0"])[seg]; T = np.array(vals["a_T1_T2_ms"])[seg] * 1e-3
    pha = phantom(y=ys, M0=M0, T1=T, T2=T)
    # (b) two concentric discs
    g = (np.arange(120) + 0.5) * 1e-3 - 0.06
    X, Y = np.meshgrid(g, g, indexing="ij")
    rr = np.hypot(X, Y).ravel()
    keep = rr <= vals["b_R_mm"][0] * 1e-3
    inner = rr[keep] <= vals["b_r_mm"][0] * 1e-3
    Tb = np.where(inner, vals["b_T_inner_ms"][0], vals["b_T_outer_ms"][0]) * 1e-3
    dwb = np.where(inner, vals["b_dw_inner_rad_s"][0], 0.0)
    phb = phantom(x=X.ravel()[keep], y=Y.ravel()[keep], M0=1.0, T1=Tb, T2=Tb, dw=dwb)
    th, tp, TE = math.radians(90.0), 1e-9, 0.1          # TE = 100 ms as in the paper's EPI
    # balanced bipolar gradient so that k(TE) = 0 exactly
    tv = np.array([1e-3, 1.1e-3, 2e-3, 2.1e-3, 2.2e-3, 3.1e-3, 3.2e-3])
    gv = np.array([0, 5e-3, 5e-3, 0, -5e-3, -5e-3, 0.0])
    s = seq(g={0: (tv, gv), 1: (tv, -gv)}, rf=([0.0], [tp], [th / (GAMMA * tp)], [0.0]), adc=[TE + tp],
            t_end=TE + 1e-3, dt_rf_max=tp)
    for p in (pha, phb):
        sig = oracle_mod.simulate(p, s)
        want = 1j * math.sin(th) * np.sum(p.M0 * np.exp(-TE / p.T2) * np.exp(-1j * p.dw * TE))
        assert abs(sig[0] - want) < 1e-6 * abs(want) + 1e-9


# ---------------------------------------------------------------------------------------------- P9
def _rand_case(seed, n_sp=12):
    rng = np.random.default_rng(seed)
    ph = phantom(rng.uniform(-0.1, 0.1, n_sp), rng.uniform(-0.1, 0.1, n_sp), rng.uniform(-0.01, 0.01, n_sp),
                 rng.uniform(0.2, 1, n_sp), rng.uniform(0.3, 2, n_sp), rng.uniform(0.03, 0.2, n_sp),
                 rng.normal(0, 300, n_sp))
    n_rf, dt = 40, 5e-6
    rf_t = 50e-6 + np.arange(n_rf) * dt
    b1 = (rng.normal(0, 20e-6, n_rf) + 1j * rng.normal(0, 20e-6, n_rf))
    g = {}
    for a in range(3):
        tv = np.sort(rng.uniform(300e-6, 3e-3, 9))
        tv = np.concatenate([[10e-6, 40e-6, 260e-6, 290e-6], tv])
        gv = np.concatenate([[0, 4e-3, 4e-3, 0], rng.normal(0, 6e-3, 9)])
        gv[-1] = 0.0
        gv[4] = 0.0
        g[a] = (tv, gv)
    adc = np.sort(rng.uniform(300e-6, 3.2e-3, 25))
    return ph, dict(g=g, rf=(rf_t, np.full(n_rf, dt), b1.real, b1.imag), adc=adc, t_end=3.5e-3, dt_rf_max=dt)


def test_p9_linearity_superposition_and_norm(oracle_mod):
    ph, kw = _rand_case(9)
    s = seq(**kw)
    full = oracle_mod.simulate(ph, s)
    a = oracle_mod.simulate(ph.subset(slice(0, 5)), s)
    b = oracle_mod.simulate(ph.subset(slice(5, None)), s)
    np.testing.assert_allclose(full, a + b, rtol=0, atol=1e-12)            # I3 superposition
    ph2 = phantom(ph.x, ph.y, ph.z, 3.0 * ph.M0, ph.T1, ph.T2, ph.dw)
    np.testing.assert_allclose(oracle_mod.simulate(ph2, s), 3.0 * full, rtol=0, atol=1e-11)   # I3 linearity
    ph3 = phantom(ph.x, ph.y, ph.z, ph.M0, 1e30, 1e30, ph.dw)
    _, mxy, mz = oracle_mod.simulate(ph3, s, return_state=True)
    np.testing.assert_allclose(np.sqrt(np.abs(mxy) ** 2 + mz ** 2), ph.M0, rtol=0, atol=1e-12)  # I1/I2


def test_p9_refinement_and_regime_switch_invariance(oracle_mod):
    ph, kw = _rand_case(10)
    base = oracle_mod.simulate(ph, seq(**kw))
    # I4: extra points in RF-free intervals (linearly interpolated G) change nothing
    kw2 = dict(kw)
    g2 = {}
    for a, (tv, gv) in kw["g"].items():
        extra = np.linspace(300e-6, 3.4e-3, 333)
        tt = np.union1d(tv, extra)
        g2[a] = (tt, np.interp(tt, tv, gv, left=0.0, right=0.0))
    kw2["g"] = g2
    np.testing.assert_allclose(oracle_mod.simulate(ph, seq(**kw2)), base, rtol=0, atol=1e-11)
    # I5: RF-free intervals forced through the excitation branch equal the precession branch
    forced = oracle_mod.simulate(ph, seq(**kw), force_excitation=True)
    np.testing.assert_allclose(forced, base, rtol=0, atol=1e-11)


def test_p9_b1_phase_and_translation(oracle_mod):
    ph, kw = _rand_case(11)
    s = seq(**kw)
    base = oracle_mod.simulate(ph, s)
    psi = 0.7
    rf_t, rf_dt, re, im = kw["rf"]
    b = (re + 1j * im) * np.exp(1j * psi)
    kw2 = dict(kw); kw2["rf"] = (rf_t, rf_dt, b.real, b.imag)
    np.testing.assert_allclose(oracle_mod.simulate(ph, seq(**kw2)), base * np.exp(1j * psi), rtol=0, atol=1e-11)  # I6
    # I7: translation by d multiplies S(t) by exp(-i 2 pi k(t).d) -- only when no gradient plays during RF
    kw3 = dict(kw)
    kw3["g"] = {a: (tv[4:], np.concatenate([[0.0], gv[5:]])) for a, (tv, gv) in kw["g"].items()}
    s3 = seq(**kw3)
    base3 = oracle_mod.simulate(ph, s3)
    d = np.array([0.004, -0.007, 0.002])
    ph_t = phantom(ph.x + d[0], ph.y + d[1], ph.z + d[2], ph.M0, ph.T1, ph.T2, ph.dw)
    moved = oracle_mod.simulate(ph_t, s3)
    k = np.zeros((len(kw["adc"]), 3))
    for a, (tv, gv) in kw3["g"].items():
        for j, t in enumerate(kw["adc"]):
            tt = np.union1d(tv[tv < t], [t])
            k[j, a] = np.trapezoid(np.interp(tt, tv, gv, left=0.0, right=0.0), tt) * GAMMA / (2 * math.pi)
    np.testing.assert_allclose(moved, base3 * np.exp(-2j * math.pi * (k @ d)), rtol=0, atol=1e-10)


# ---------------------------------------------------------------------------------------------- P10
def test_p10_second_order_global_convergence(oracle_mod):
    T, tbw = 1e-3, 4.0
    ph = phantom(z=np.linspace(-6e-3, 6e-3, 9), T1=0.5, T2=0.05)
    gz = 4.0 / (T * 42.58e6 * 5e-3)

    def run(n):
        dt = T / n
        tm = (np.arange(n) + 0.5) * dt
        env = np.sinc(tbw * (tm - T / 2) / T)
        b1 = env * (math.radians(70.0) / (GAMMA * dt * env.sum()))
        s = seq(g={2: (np.array([0.0, 100e-6, 100e-6 + T, 200e-6 + T]), np.array([0, gz, gz, 0.0]))},
                rf=(100e-6 + np.arange(n) * dt, np.full(n, dt), b1, np.zeros(n)), t_end=200e-6 + T,
                dt_rf_max=dt)
        _, mxy, mz = oracle_mod.simulate(ph, s, return_state=True)
        return np.concatenate([mxy.real, mxy.imag, mz])

    r = [run(n) for n in (50, 100, 200, 400)]
    d1, d2, d3 = (np.abs(r[i + 1] - r[i]).max() for i in range(3))
    assert 3.3 < d1 / d2 < 4.7 and 3.3 < d2 / d3 < 4.7       # global O(dt^2) from local O(dt^3)


# ------------------------------------------------------------------------------ discretiser (a1) pins
def test_grid_contents_and_rf_refinement(oracle_mod):
    s = seq(g={0: ([1e-3, 2e-3, 3e-3], [0, 1e-3, 0])}, rf=([0.0], [0.5e-3], [1e-6], [0.0]),
            adc=[1.5e-3, 2.5e-3], t_end=4e-3, dt_rf_max=0.1e-3)
    t, G, rf, adc = oracle_mod.grid(s)
    want_t = np.concatenate([np.arange(6) * 0.1e-3, [1e-3, 1.5e-3, 2e-3, 2.5e-3, 3e-3, 4e-3]])
    np.testing.assert_allclose(t, want_t, rtol=0, atol=1e-15)
    assert rf.tolist() == [1] * 5 + [0] * 6
    np.testing.assert_allclose(G[:, 0], np.interp(want_t, [1e-3, 2e-3, 3e-3], [0, 1e-3, 0]), atol=1e-18)
    assert adc.tolist() == [-1] * 7 + [0, -1, 1, -1, -1]


@pytest.mark.parametrize("t0", [0.0, 0.7300001, 12.000123, 14.9876543])
def test_rf_train_late_in_a_long_sequence_keeps_its_nominal_step_count(oracle_mod, t0):
    """Reading G18, pinned by counting: an RF train of 1000 samples of nominal 1 us with
    dt_rf_max = 1 us is 1000 RF intervals wherever it sits on the time axis.  At t ~ 12 s the spacing of doubles is
    1.8e-15 s, so rf_t[i+1] - rf_t[i] exceeds 1e-6 by rounding for about a third of the samples; a refinement rule
    without the 1e-12 s time tolerance (reading G13) cuts those in two (it did: 362 of config 5's 1000 TRs).  A piece
    that really is longer than dt_rf_max -- by more than the tolerance -- is still cut."""
    n, dt = 1000, 1e-6
    rf_t = t0 + np.arange(n) * dt
    s = seq(rf=(rf_t, np.full(n, dt), np.full(n, 1e-6), np.zeros(n)), t_end=t0 + n * dt + 1e-3, dt_rf_max=dt)
    t, _, rf, _ = oracle_mod.grid(s)
    assert int(rf.sum()) == n                                   # the nominal count, not n + (rounding splits)
    steps = np.diff(t)[rf.astype(bool)]
    assert steps.min() > 0.99 * dt and steps.max() < 1.01 * dt  # and no half steps hide in it
    # the physics agrees: the train's flip angle on resonance is gamma * B1 * n * dt whatever the grid (P3), so the
    # count is the only thing this reading can change -- and the count is what the benchmark's spin*steps are made of
    # genuinely longer pieces are cut: 2.5 us -> 3 sub-steps, 1 us + 5e-12 s -> 2
    for dur, parts in ((2.5e-6, 3), (1e-6 + 5e-12, 2), (1e-6 + 5e-13, 1)):
        s2 = seq(rf=([t0 + 1e-4], [dur], [1e-6], [0.0]), t_end=t0 + 1e-3, dt_rf_max=dt)
        assert int(oracle_mod.grid(s2)[2].sum()) == parts


# ---------------------------------------------------------------------------------------------- f2
def test_grouped_output_is_a_fisp_ensemble_dictionary(oracle_mod):
    """three (T1, T2) entries, each an ensemble of 128 isochromats whose spoiler phase covers
    2 pi per TR; the grouped signal of entry g, divided by the group size, must be ITS closed-form FISP FID
    steady state (P7 formula) -- which pins the group indexing and ordering, not only the sum.  Degenerate
    group sizes reduce to the other two modes."""
    alpha, TR, n_iso, n_tr = math.radians(30.0), 6e-3, 128, 300
    T1s, T2s = np.array([0.1, 0.25, 0.08]), np.array([0.04, 0.02, 0.06])
    tp = 1e-9
    rf_t = np.arange(n_tr) * TR
    s = seq(rf=(rf_t, np.full(n_tr, tp), np.full(n_tr, alpha / (GAMMA * tp)), np.zeros(n_tr)),
            adc=[rf_t[-1] + tp], t_end=rf_t[-1] + TR, dt_rf_max=tp)
    dws = np.tile(2 * math.pi * np.arange(n_iso) / (n_iso * TR), 3)
    ph = phantom(M0=1.0, T1=np.repeat(T1s, n_iso), T2=np.repeat(T2s, n_iso), dw=dws)
    grouped = oracle_mod.simulate(ph, s, output_mode="grouped", group_size=n_iso)
    assert grouped.shape == (3, 1)
    ca = math.cos(alpha)
    for g in range(3):
        E1, E2 = math.exp(-TR / T1s[g]), math.exp(-TR / T2s[g])
        r = math.sqrt((1 - E2 ** 2) / ((1 - E1 * ca) ** 2 - E2 ** 2 * (E1 - ca) ** 2))
        fid = math.tan(alpha / 2) * (1 - (E1 - ca) * r)
        assert abs(abs(grouped[g, 0]) / n_iso - fid) < 1e-6, g
    per = oracle_mod.simulate(ph, s, output_mode="per_spin")
    np.testing.assert_allclose(oracle_mod.simulate(ph, s, output_mode="grouped", group_size=1), per, rtol=0, atol=0)
    total = oracle_mod.simulate(ph, s)
    np.testing.assert_allclose(oracle_mod.simulate(ph, s, output_mode="grouped", group_size=3 * n_iso)[0], total,
                               rtol=0, atol=1e-10)
    with pytest.raises(ValueError):
        oracle_mod.simulate(ph, s, output_mode="grouped", group_size=5)


# ---------------------------------------------------------------------------------------------- P11
def hs_pulse(T, n, w1max, mu, beta, t0=0.0):
    """Hyperbolic-secant pulse B1(t) = (w1max / gamma) sech(beta t)^(1 + i mu), piecewise constant at step midpoints."""
    dt = T / n
    tm = (np.arange(n) + 0.5) * dt - T / 2
    amp = w1max / GAMMA / np.cosh(beta * tm)
    phi = mu * np.log(1.0 / np.cosh(beta * tm))
    return t0 + np.arange(n) * dt, np.full(n, dt), amp * np.cos(phi), amp * np.sin(phi)


@pytest.mark.parametrize("w1max", [3000.0, 4500.0])
def test_p11_adiabatic_hyperbolic_secant_inversion_profile(oracle_mod, w1max):
    """A long soft pulse with a frequency sweep -- the paper's own weak spot ("long soft RF pulses
    (like adiabatic pulses)") -- has a closed form without relaxation: for B1 = w1max sech(beta t)^(1+i mu) over the
    whole time axis the Bloch equations solve in hypergeometric functions and
        Mz/M0 = tanh(a+b) tanh(a-b) + cos(pi sqrt((w1max/beta)^2 - mu^2)) sech(a+b) sech(a-b),
        a = pi Omega / (2 beta), b = pi mu / 2                       (Silver, Joseph & Hoult, Phys Rev A 31, 1985).
    15,000 steps of complex, phase-modulated B1 composed by Eq 6-9 must land on it for every off-resonance Omega,
    inside, on the edge of and outside the inverted band |Omega| < mu beta; the pulse is cut at beta T/2 = 12 where
    sech = 1.2e-5.  Both amplitudes (below and above w1max = mu beta, where the square root turns imaginary)."""
    mu, beta, T, n = 5.0, 800.0, 30e-3, 15000
    Om = np.linspace(-8000.0, 8000.0, 81)
    ph = phantom(dw=Om)                                            # T1 = T2 = inf
    s = seq(rf=hs_pulse(T, n, w1max, mu, beta), t_end=T, dt_rf_max=T / n)
    _, mxy, mz = oracle_mod.simulate(ph, s, return_state=True)
    a, b = math.pi * Om / (2 * beta), math.pi * mu / 2
    root = np.sqrt(complex((w1max / beta) ** 2 - mu ** 2))
    want = np.tanh(a + b) * np.tanh(a - b) + np.cos(math.pi * root).real / (np.cosh(a + b) * np.cosh(a - b))
    np.testing.assert_allclose(mz, want, rtol=0, atol=1e-4)
    np.testing.assert_allclose(np.abs(mxy) ** 2 + mz ** 2, 1.0, rtol=0, atol=1e-9)   # a rotation: |M| kept
    inside, outside = np.abs(Om) < 0.4 * mu * beta, np.abs(Om) > 1.5 * mu * beta
    assert mz[inside].max() < -0.98 and mz[outside].min() > 0.999                      # what "inversion band" means


# ---------------------------------------------------------------------------------------------- P12
def test_p12_frequency_offset_pulse_excites_the_shifted_slice(oracle_mod):
    """Reading G12 (B1 is complex; an RF frequency offset is a phase ramp on it) together with reading G3 (free
    precession is Mxy e^{-i dw t}): a pulse B1(t) e^{-i 2 pi df t} under a slice gradient Gz is, in the frame rotating
    at df, the same pulse on resonance for the spin at z0 = df / (gamma_bar Gz).  So the excited profile is the
    on-centre profile moved to z0 -- same Mz, same |Mxy| -- and NOT to -z0 (which is what a sign slip between the
    B1 phase convention and the precession direction would give).  PAPER.md:99-101 off-centre slices."""
    T, n, Gz, df = 2e-3, 4000, 8e-3, 3000.0     # 0.5 us steps: the piecewise-constant phase ramp costs (2 pi df dt)^2 / 24 = 4e-6
    dt = T / n
    tm = (np.arange(n) + 0.5) * dt
    env = np.sinc(4.0 * (tm - T / 2) / T) * (0.54 + 0.46 * np.cos(2 * math.pi * (tm - T / 2) / T))
    b1 = env * (math.pi / 3) / (GAMMA * dt * env.sum())
    z0 = df / (GAMMA / (2 * math.pi) * Gz)                     # 8.8 mm
    z = np.linspace(-0.02, 0.02, 161)
    g = {2: ([0.0, T], [Gz, Gz])}
    on = seq(g=g, rf=(np.arange(n) * dt, np.full(n, dt), b1, np.zeros(n)), t_end=T, dt_rf_max=dt)
    ph = -2 * math.pi * df * tm
    off = seq(g=g, rf=(np.arange(n) * dt, np.full(n, dt), b1 * np.cos(ph), b1 * np.sin(ph)), t_end=T, dt_rf_max=dt)
    _, mxy_on, mz_on = oracle_mod.simulate(phantom(z=z - z0), on, return_state=True)     # profile at z' = z - z0
    _, mxy_off, mz_off = oracle_mod.simulate(phantom(z=z), off, return_state=True)
    np.testing.assert_allclose(mz_off, mz_on, rtol=0, atol=2e-5)
    np.testing.assert_allclose(np.abs(mxy_off), np.abs(mxy_on), rtol=0, atol=2e-5)
    # in the frame rotating at df the transverse magnetisation is the on-centre one: Mxy_off = Mxy_on e^{-i 2 pi df T}
    np.testing.assert_allclose(mxy_off, mxy_on * np.exp(-2j * math.pi * df * T), rtol=0, atol=2e-5)
    # and the slice really sits at +z0: the profile's centre of mass
    com = (z * np.abs(mxy_off)).sum() / np.abs(mxy_off).sum()
    assert abs(com - z0) < 2e-4 and np.abs(mxy_off)[np.argmin(np.abs(z + z0))] < 0.02
