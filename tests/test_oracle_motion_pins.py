"""Pins for the oracle's motion extension (PAPER.md:96 motion field u(x,t), :180
intermediate points "in the case of motion", :236 experiment (d) u_y = v_y t): x(t) = x + v t per spin.
None of these call the CUDA path."""
import numpy as np
import pytest

from seqtools import phantom, seq

GAMMA = 2.0 * np.pi * 42.58e6


def run(oracle_mod, ph, s, v, state=None, **kw):
    if state is None:
        state = (np.ones(ph.x.shape[0], dtype=np.complex128), np.zeros(ph.x.shape[0]))
    return oracle_mod.simulate(ph, s, state=state, velocity=v, output_mode="per_spin", **kw)


def test_m1_constant_gradient_constant_velocity_closed_form(oracle_mod):
    """G constant, x(t) = x0 + v t: G.x(t) is linear in t, so the trapezoid on ANY grid is exact and
    Mxy(t) = exp(-i gamma G (x0 t + v t^2 / 2)) exp(-i dw t) exp(-t/T2)."""
    G, T = 7e-3, 4e-3
    x0 = np.array([0.01, -0.03, 0.05])
    v = np.array([0.1, -0.25, 0.0])
    dw = np.array([30.0, 0.0, -80.0])
    adc = np.array([0.3e-3, 1.1e-3, 2.7e-3, 4e-3])
    s = seq(g={1: ([0.0, T], [G, G])}, adc=adc, t_end=T)
    ph = phantom(y=x0, T2=[0.05, 0.1, 1e30], dw=dw)
    sig = run(oracle_mod, ph, s, (np.zeros(3), v, np.zeros(3)))
    for i in range(3):
        exact = np.exp(-1j * (GAMMA * G * (x0[i] * adc + v[i] * adc ** 2 / 2) + dw[i] * adc)) * np.exp(-adc / ph.T2[i])
        np.testing.assert_allclose(sig[i], exact, rtol=0, atol=2e-11)
    # refining the grid changes nothing here (exactness), and zero velocity equals the static entry
    sig2 = run(oracle_mod, ph, s, (np.zeros(3), v, np.zeros(3)), dt_max=1e-5)
    np.testing.assert_allclose(sig2, sig, rtol=0, atol=2e-11)
    stat = oracle_mod.simulate(ph, s, state=(np.ones(3, dtype=np.complex128), np.zeros(3)), output_mode="per_spin")
    zero = run(oracle_mod, ph, s, (np.zeros(3), np.zeros(3), np.zeros(3)))
    np.testing.assert_allclose(zero, stat, rtol=0, atol=1e-14)


def test_m2_bipolar_pair_encodes_velocity_not_position(oracle_mod):
    """Rectangular bipolar lobes (+G for d, -G for d): zeroth moment 0, first moment -G d^2, so the phase after
    the pair is +gamma v G d^2 whatever x0 is (velocity encoding).  The lobes are given with 1 ns edges; the
    trapezoid on the edge intervals carries an O(edge) error, far below the tolerance used."""
    G, d, e = 10e-3, 1e-3, 1e-9
    t0 = 0.5e-3
    tv = [t0, t0 + e, t0 + d, t0 + d + e, t0 + 2 * d, t0 + 2 * d + e]
    gv = [0.0, G, G, -G, -G, 0.0]
    adc = [t0 + 2 * d + 1e-4]
    s = seq(g={0: (tv, gv)}, adc=adc, t_end=3e-3)
    x0 = np.array([-0.04, 0.0, 0.07, 0.07])
    v = np.array([0.1, 0.1, 0.1, -0.3])
    sig = run(oracle_mod, phantom(x=x0), s, (v, np.zeros(4), np.zeros(4)))[:, 0]
    expected = np.exp(1j * GAMMA * v * G * d * d)
    np.testing.assert_allclose(sig, expected, rtol=0, atol=5e-5)
    assert abs(sig[0] - sig[2]) < 1e-4            # same v, different x0
    static = run(oracle_mod, phantom(x=x0), s, (np.zeros(4), np.zeros(4), np.zeros(4)))[:, 0]
    np.testing.assert_allclose(static, np.ones(4), rtol=0, atol=5e-5)


def test_m3_a_ramp_converges_with_dt_max_at_second_order(oracle_mod):
    """On a ramp G(t).x(t) is quadratic in t, so the trapezoid needs the intermediate points of :180; halving
    dt_max must shrink the error about 4x towards the analytic moment.  A single sawtooth ramp is used: on a
    symmetric trapezoid lobe the errors of the up and down ramps cancel exactly."""
    G, R, e, t0 = 12e-3, 1e-3, 1e-9, 2e-4
    s = seq(g={2: ([t0, t0 + R, t0 + R + e], [0.0, G, 0.0])}, adc=[t0 + R + 1e-4], t_end=2e-3)
    v = 0.2
    m1 = G * (R * R / 3 + t0 * R / 2)              # int G(t) t dt over the ramp, x0 = 0
    exact = np.exp(-1j * GAMMA * v * m1)
    errs = []
    for dt in (4e-5, 2e-5, 1e-5):
        sig = run(oracle_mod, phantom(z=[0.0]), s, (np.zeros(1), np.zeros(1), np.array([v])), dt_max=dt)[0, 0]
        errs.append(abs(sig - exact))
    assert errs[0] > 1e-5, "coarse grid should show the trapezoid error"
    assert 3.7 < errs[0] / errs[1] < 4.3 and 3.7 < errs[1] / errs[2] < 4.3, errs


def test_m4_both_regimes_see_the_same_moving_field(oracle_mod):
    """Invariant I5 with motion: RF-free intervals pushed through the excitation branch give the precession
    branch's answer, so both branches use the same Bz for a moving spin."""
    rng = np.random.default_rng(3)
    n = 6
    ph = phantom(x=rng.uniform(-.1, .1, n), y=rng.uniform(-.1, .1, n), z=rng.uniform(-.1, .1, n),
                 T1=rng.uniform(.3, 2, n), T2=rng.uniform(.03, .3, n), dw=rng.uniform(-200, 200, n))
    v = tuple(rng.uniform(-.3, .3, n) for _ in range(3))
    g = {0: ([0, 1e-3, 2e-3], [0, 8e-3, -3e-3]), 1: ([2e-4, 1.5e-3], [5e-3, 0]), 2: ([0, 2e-3], [-4e-3, 6e-3])}
    s = seq(g=g, adc=np.linspace(1e-4, 2e-3, 9), t_end=2e-3)
    st = (rng.normal(size=n) + 1j * rng.normal(size=n), rng.normal(size=n))
    a = oracle_mod.simulate(ph, s, state=st, velocity=v, dt_max=2e-5, output_mode="per_spin")
    b = oracle_mod.simulate(ph, s, state=st, velocity=v, dt_max=2e-5, output_mode="per_spin", force_excitation=True)
    np.testing.assert_allclose(a, b, rtol=0, atol=1e-12)


def test_m5_dt_max_refines_every_interval(oracle_mod):
    s = seq(g={0: ([0.0, 1e-3], [0.0, 5e-3])}, rf=([2e-4], [1e-4], [1e-6], [0.0]), adc=[5e-4], t_end=1e-3,
            dt_rf_max=2e-5)
    t0, *_ = oracle_mod.grid(s)
    t1, _, rf1, _ = oracle_mod.grid(s, dt_max=5e-5)
    assert len(t1) > len(t0) and np.diff(t1).max() <= 5e-5 + 1e-12
    assert np.all(np.diff(t1)[rf1.astype(bool)] <= 2e-5 + 1e-12)
    t2, *_ = oracle_mod.grid(s, dt_max=1e-5)       # dt_max below dt_rf_max also limits RF steps
    assert np.diff(t2).max() <= 1e-5 + 1e-12


# ------------------------------------------------------------------------------------------------------------------
# General motion ("motion field u(x, t)"; reading M2): x(t) = x + a u(t), a per spin, u(t) a shared
# piecewise-linear waveform.  Pins W1-W5.
# ------------------------------------------------------------------------------------------------------------------
def runw(oracle_mod, ph, s, a, wf, **kw):
    state = (np.ones(ph.x.shape[0], dtype=np.complex128), np.zeros(ph.x.shape[0]))
    return oracle_mod.simulate(ph, s, state=state, velocity=a, waveform=wf, output_mode="per_spin", **kw)


def test_w1_sinusoidal_displacement_under_a_constant_gradient_closed_form(oracle_mod):
    """G constant, x(t) = x0 + a u(t) with u the piecewise-linear interpolant of sin(2 pi f t) on 65 vertices:
    G.x(t) is piecewise linear between the waveform's vertices, which are points of the grid, so the trapezoid is EXACT
    and the phase at time t is -gamma G (x0 t + a U(t)), U(t) the exact integral of the interpolant; against the
    analytic sinusoid the difference is the interpolation error of the waveform only (O(h^2))."""
    G, T, f = 5e-3, 8e-3, 250.0
    wt = np.linspace(0.0, T, 65)
    wu = np.sin(2 * np.pi * f * wt)
    x0 = np.array([0.02, -0.01, 0.0])
    a = np.array([2e-3, -5e-3, 1e-3])          # displacement amplitudes [m]
    adc = np.array([0.7e-3, 2.0e-3, 3.3e-3, 6.1e-3, 8e-3])
    s = seq(g={0: ([0.0, T], [G, G])}, adc=adc, t_end=T)
    sig = runw(oracle_mod, phantom(x=x0), s, (a, np.zeros(3), np.zeros(3)), (wt, wu))

    def U(t):  # exact integral of the piecewise-linear interpolant from 0 to t
        tt = np.union1d(wt[wt < t], [t])
        return np.trapezoid(np.interp(tt, wt, wu), tt)

    for i in range(3):
        exact = np.exp(-1j * GAMMA * G * np.array([x0[i] * t + a[i] * U(t) for t in adc]))
        np.testing.assert_allclose(sig[i], exact, rtol=0, atol=5e-11)
        analytic = np.exp(-1j * GAMMA * G * (x0[i] * adc + a[i] * (1 - np.cos(2 * np.pi * f * adc)) / (2 * np.pi * f)))
        assert np.abs(sig[i] - analytic).max() < 5e-2      # waveform interpolation error (O(h^2)), not the integrator's
    wt8 = np.linspace(0.0, T, 513)                          # 8 x finer vertices: 64 x closer to the analytic sinusoid
    fine = runw(oracle_mod, phantom(x=x0), s, (a, np.zeros(3), np.zeros(3)), (wt8, np.sin(2 * np.pi * f * wt8)))
    for i in range(3):
        analytic = np.exp(-1j * GAMMA * G * (x0[i] * adc + a[i] * (1 - np.cos(2 * np.pi * f * adc)) / (2 * np.pi * f)))
        assert np.abs(fine[i] - analytic).max() < 1e-3
    # exactness: a finer grid changes nothing
    sig2 = runw(oracle_mod, phantom(x=x0), s, (a, np.zeros(3), np.zeros(3)), (wt, wu), dt_max=2e-5)
    np.testing.assert_allclose(sig2, sig, rtol=0, atol=5e-11)


def test_w2_waveform_u_equal_t_is_the_constant_velocity_entry(oracle_mod):
    """u(t) = t given as a two-vertex waveform reproduces x(t) = x + v t (pins M1-M5 then carry over): with RF, a ramp
    and dt_max refinement, signal and final state agree to rounding."""
    rng = np.random.default_rng(3)
    n = 6
    ph = phantom(x=rng.uniform(-.05, .05, n), y=rng.uniform(-.05, .05, n), z=rng.uniform(-.01, .01, n),
                 T1=rng.uniform(.3, 2, n), T2=rng.uniform(.03, .3, n), dw=rng.uniform(-200, 200, n))
    v = tuple(rng.uniform(-0.3, 0.3, n) for _ in range(3))
    rf = (np.arange(40) * 5e-6, np.full(40, 5e-6), np.full(40, 4e-6), np.linspace(-1e-6, 1e-6, 40))
    g = {0: ([0, 2e-4, 1.5e-3, 1.7e-3], [0, 6e-3, -4e-3, 0]), 2: ([0, 1e-5, 1.9e-4, 2e-4], [0, 8e-3, 8e-3, 0])}
    s = seq(g=g, rf=rf, adc=2.5e-4 + np.arange(30) * 4e-5, t_end=2e-3, dt_rf_max=5e-6)
    ref = oracle_mod.simulate(ph, s, velocity=v, dt_max=2e-5, output_mode="per_spin", return_state=True)
    got = oracle_mod.simulate(ph, s, velocity=v, dt_max=2e-5, output_mode="per_spin", return_state=True,
                              waveform=([0.0, 2e-3], [0.0, 2e-3]))
    for a, b in zip(got, ref):
        np.testing.assert_allclose(a, b, rtol=0, atol=1e-12)


def test_w3_stop_and_go_only_the_displaced_position_counts_while_u_is_flat(oracle_mod):
    """u ramps from 0 to 1 during [1, 2] ms and stays there: a gradient lobe played while u is flat sees a spin at rest
    at x0 + a (phase -gamma area (x0 + a)), one played before the move sees x0; amplitudes beyond the last vertex keep
    the end value (no extrapolation)."""
    wf = ([1e-3, 2e-3], [0.0, 1.0])
    area_t = [2.5e-3, 2.6e-3, 3.4e-3, 3.5e-3]
    early_t = [0.0e-3, 0.1e-3, 0.9e-3, 1.0e-3]
    Gp = 6e-3
    x0 = np.array([0.01, -0.02])
    a = np.array([4e-3, -7e-3])
    area = Gp * 0.9e-3
    for tv, pos in ((area_t, x0 + a), (early_t, x0)):
        s = seq(g={1: (tv, [0, Gp, Gp, 0])}, adc=[4e-3], t_end=4e-3)
        sig = runw(oracle_mod, phantom(y=x0), s, (np.zeros(2), a, np.zeros(2)), wf, dt_max=1e-5)[:, 0]
        np.testing.assert_allclose(sig, np.exp(-1j * GAMMA * area * pos), rtol=0, atol=1e-10)


def test_w4_a_periodic_displacement_that_returns_leaves_no_trace_on_a_later_echo(oracle_mod):
    """A displacement that has returned to zero before a gradient pair is played does not change what that pair does:
    the signal after the pair equals the static one; with the pair played DURING the excursion it does not."""
    wt = np.linspace(0.0, 2e-3, 41)
    wu = np.sin(np.pi * wt / 2e-3) ** 2            # out and back, 0 at both ends
    G, d = 8e-3, 0.5e-3
    a = np.array([3e-3, -2e-3, 5e-3])
    x0 = np.array([0.03, 0.0, -0.02])

    def pair(t0):
        e = 1e-8
        return [t0, t0 + e, t0 + d, t0 + d + e, t0 + 2 * d, t0 + 2 * d + e], [0.0, G, G, -G, -G, 0.0]

    for t0, moved in ((2.2e-3, False), (0.1e-3, True)):   # 0.1 .. 1.1 ms: the rising half of the excursion
        tv, gv = pair(t0)
        s = seq(g={0: (tv, gv)}, adc=[3.5e-3], t_end=3.6e-3)
        mov = runw(oracle_mod, phantom(x=x0), s, (a, np.zeros(3), np.zeros(3)), (wt, wu), dt_max=1e-5)[:, 0]
        stat = oracle_mod.simulate(phantom(x=x0), s, state=(np.ones(3, dtype=np.complex128), np.zeros(3)),
                                   output_mode="per_spin")[:, 0]
        if moved:
            assert np.abs(mov - stat).min() > 1e-2
        else:
            np.testing.assert_allclose(mov, stat, rtol=0, atol=1e-9)


def test_w5_second_order_convergence_in_dt_max_under_a_ramp(oracle_mod):
    """G(t) = s t (a ramp) and u(t) = t^2-like piecewise-linear waveform with many vertices: G.x(t) is no longer
    piecewise linear between grid points, the trapezoid converges at O(dt_max^2) to the integral of the product."""
    T, slew = 2e-3, 3.0
    wt = np.linspace(0.0, T, 5)
    wu = (wt / T) ** 2
    a = np.array([6e-3])
    s = seq(g={0: ([0.0, T], [0.0, slew * T])}, adc=[T], t_end=T)
    # exact integral of G(t) a u(t) with u the piecewise-linear interpolant: piecewise cubic, by Simpson per piece
    tt = np.linspace(0.0, T, 5)
    exact_int = 0.0
    for k in range(4):
        t0, t1 = tt[k], tt[k + 1]
        f = lambda t: slew * t * np.interp(t, wt, wu)
        exact_int += (t1 - t0) / 6 * (f(t0) + 4 * f(0.5 * (t0 + t1)) + f(t1))      # exact for a quadratic integrand
    exact = np.exp(-1j * GAMMA * a[0] * exact_int)
    errs = []
    for dt in (2.5e-4, 1.25e-4, 6.25e-5):     # 2, 4, 8 equal sub-steps of every 0.5 ms piece between waveform vertices
        sig = runw(oracle_mod, phantom(x=[0.0]), s, (a, np.zeros(1), np.zeros(1)), (wt, wu), dt_max=dt)[0, 0]
        errs.append(abs(sig - exact))
    assert errs[0] > errs[1] > errs[2]
    assert 3.3 < errs[0] / errs[1] < 4.7 and 3.3 < errs[1] / errs[2] < 4.7


def test_waveform_vertices_join_the_grid_and_bad_waveforms_are_rejected(oracle_mod):
    s = seq(g={0: ([0.0, 1e-3], [1e-3, 1e-3])}, adc=[5e-4], t_end=1e-3)
    t, _, _, _ = oracle_mod.grid(s, waveform=([2e-4, 3.3e-4, 7e-4], [0.0, 1.0, 0.0]))
    np.testing.assert_allclose(t, [0.0, 2e-4, 3.3e-4, 5e-4, 7e-4, 1e-3], rtol=0, atol=1e-15)
    with pytest.raises(ValueError):
        oracle_mod.grid(s, waveform=([3e-4, 2e-4], [0.0, 1.0]))          # not ascending
    with pytest.raises(ValueError):
        oracle_mod.simulate(phantom(), s, waveform=([0.0, 1e-3], [0.0, 1.0]))   # amplitudes missing
