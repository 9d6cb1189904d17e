"""GPU-vs-oracle parity with moving spins, x(t) = x + v t.
Same acceptance as the static path: max <= 1e-4, NRMSE <= 1e-5 of the oracle maximum."""
import numpy as np
import pytest

from paper_2301_02702_b200 import workloads as W
from seqtools import seq

pytestmark = pytest.mark.gpu

TOL_MAX = 1e-4
TOL_NRMSE = 1e-5


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2301_02702_b200 import build as bl
    bl.build()
    from paper_2301_02702_b200 import bloch
    return bloch


def errors(got, ref):
    got = np.asarray(got, dtype=np.complex128)
    ref = np.asarray(ref, dtype=np.complex128)
    scale = np.abs(ref).max()
    d = np.abs(got - ref)
    return d.max() / scale, np.sqrt(np.mean(d ** 2)) / scale


def f32(a):
    return np.asarray(a, dtype=np.float32).astype(np.float64)


def run_both(B, oracle_mod, ph, s, v, dt_max, what, output_mode="sum", phase_mode="auto", host=False, options=None,
             waveform=None, **plan_kw):
    import torch
    v = tuple(f32(a) for a in v)
    mo = dict(motion="linear") if waveform is None else dict(motion="waveform", waveform=waveform)
    plan = B.Plan(s, output_mode=output_mode, phase_mode=phase_mode, dt_max=dt_max, options=options, **mo, **plan_kw)
    assert plan.info["motion_mode"] == (1 if waveform is None else 2)
    t, *_ = oracle_mod.grid(s, dt_max=dt_max, waveform=waveform)
    assert plan.info["n_intervals"] == len(t) - 1, "planner and oracle refine the grid differently"
    if host:
        Mxy = np.zeros((ph.n, 2), dtype=np.float32)
        Mz = np.zeros(ph.n, dtype=np.float32)
        sig = plan.simulate_host(ph.x, ph.y, ph.z, ph.M0, ph.T1, ph.T2, ph.dw, Mxy=Mxy, Mz=Mz, velocity=v)
        m, z = Mxy, Mz
    else:
        dev = B.phantom_to_device(ph)
        vel = tuple(torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda() for a in v)
        Mxy = torch.zeros(ph.n, 2, dtype=torch.float32, device="cuda")
        Mz = torch.zeros(ph.n, dtype=torch.float32, device="cuda")
        sig = plan.simulate(*dev, Mxy=Mxy, Mz=Mz, velocity=vel)
        torch.cuda.synchronize()
        sig, m, z = sig.cpu().numpy(), Mxy.cpu().numpy(), Mz.cpu().numpy()
    plan.close()
    ref, rxy, rz = oracle_mod.simulate(ph, s, velocity=v, dt_max=dt_max, output_mode=output_mode, return_state=True,
                                       waveform=waveform)
    got_state = np.concatenate([m[:, 0] + 1j * m[:, 1], z.astype(np.complex128)])
    ref_state = np.concatenate([rxy, rz.astype(np.complex128)])
    for name, g, r in (("signal", sig, ref), ("state", got_state, ref_state)):
        emax, nrmse = errors(g, r)
        print(f"{what} {name}: max {emax:.3e} nrmse {nrmse:.3e}")
        assert emax <= TOL_MAX and nrmse <= TOL_NRMSE, f"{what} {name}: max {emax:.3e} nrmse {nrmse:.3e}"
    return sig, ref


def moving_phantom(n, seed):
    rng = np.random.default_rng(seed)
    ph = W._phantom(rng.uniform(-.1, .1, n), rng.uniform(-.1, .1, n), rng.uniform(-.005, .005, n),
                    rng.uniform(.5, 1, n), rng.uniform(.3, 2, n), rng.uniform(.03, .3, n), rng.uniform(-100, 100, n))
    v = (rng.uniform(-.2, .2, n), rng.uniform(-.2, .2, n), rng.uniform(-.05, .05, n))
    return ph, v


@pytest.mark.parametrize("phase_mode", ["fp32", "fp64"])
def test_epi_with_in_plane_motion_like_experiment_d(B, oracle_mod, phase_mode):
    """Config-1-like EPI (hard 90 + 32x32 readout) with every spin moving: the paper's experiment (d) has
    u_y = v_y t with v_y = 0.1 m/s (:236)."""
    w = W.small("1")
    n = w.phantom.n
    v = (np.zeros(n), np.full(n, 0.1), np.zeros(n))
    sig, ref = run_both(B, oracle_mod, w.phantom, w.seq, v, 2e-5, f"EPI v_y=0.1 {phase_mode}", phase_mode=phase_mode)
    static = oracle_mod.simulate(w.phantom, w.seq)
    assert errors(ref, static)[0] > 1e-2, "the motion must change the signal for the test to mean anything"


def test_slice_selective_rf_on_moving_spins_and_ramps(B, oracle_mod):
    """Through-plane motion during a slice-selective sinc (RF tiles with motion records), a bipolar pair on a
    second axis, readout on a third; random velocities; 1 us RF steps, dt_max = 10 us elsewhere."""
    n_rf = 400
    dt = 1e-6
    tm = (np.arange(n_rf) + 0.5) * dt
    env = np.sinc(4.0 * (tm - n_rf * dt / 2) / (n_rf * dt))
    b1 = env * np.deg2rad(60) / (W.GAMMA * dt * env.sum())
    rf = (2e-4 + np.arange(n_rf) * dt, np.full(n_rf, dt), b1, np.zeros(n_rf))
    g = {2: ([1e-4, 2e-4, 6e-4, 7e-4, 9e-4, 1e-3], [0, 15e-3, 15e-3, 0, -12e-3, 0]),
         1: ([1.0e-3, 1.1e-3, 1.5e-3, 1.6e-3, 1.7e-3, 2.1e-3, 2.2e-3], [0, 20e-3, 20e-3, 0, -20e-3, -20e-3, 0]),
         0: ([2.2e-3, 2.3e-3, 3.6e-3, 3.7e-3], [0, 6e-3, 6e-3, 0])}
    adc = 2.3e-3 + (np.arange(321) + 0.5) * 4e-6
    s = seq(g=g, rf=rf, adc=adc, t_end=4e-3, dt_rf_max=dt)
    ph, v = moving_phantom(1500, 21)
    run_both(B, oracle_mod, ph, s, v, 1e-5, "slice-select + bipolar, moving")
    run_both(B, oracle_mod, ph, s, v, 1e-5, "same through the host entry", host=True)


def test_per_spin_output_with_motion(B, oracle_mod):
    g = {0: ([0.0, 1e-4, 2e-3], [0, 8e-3, 8e-3])}
    rf = (np.array([0.0]), np.array([5e-5]), np.array([(np.pi / 2) / (W.GAMMA * 5e-5)]), np.array([0.0]))
    adc = 2e-4 + np.arange(40) * 2e-5
    s = seq(g=g, rf=rf, adc=adc, t_end=2e-3, dt_rf_max=1.0)
    ph, v = moving_phantom(37, 22)
    run_both(B, oracle_mod, ph, s, v, 5e-5, "per-spin with motion", output_mode="per_spin")


def test_zero_velocity_equals_the_static_plan_and_velocities_need_a_motion_plan(B, oracle_mod):
    import torch
    w = W.small("4")
    n = w.phantom.n
    zero = (np.zeros(n), np.zeros(n), np.zeros(n))
    sig, _ = run_both(B, oracle_mod, w.phantom, w.seq, zero, 0.0, "zero velocity")
    plan = B.Plan(w.seq)
    dev = B.phantom_to_device(w.phantom)
    stat = plan.simulate(*dev)
    torch.cuda.synchronize()
    assert errors(sig, stat.cpu().numpy())[0] < 5e-6
    vel = tuple(torch.zeros(n, dtype=torch.float32, device="cuda") for _ in range(3))
    with pytest.raises(B.BlochError) as e:
        plan.simulate(*dev, velocity=vel)
    assert e.value.code == -1
    plan.close()


@pytest.mark.parametrize("phase_mode,n_adc", [("fp32", 2051), ("fp64", 4096)])
def test_moving_spins_on_cartesian_plateau_take_the_quadratic_recurrence(B, oracle_mod, phase_mode, n_adc):
    """>= 2048 equally spaced samples on a plateau with moving spins: k' is linear and the first moment mu' quadratic in
    the sample index, so the planner hands the block to signal_lin_kernel<., motion> (w_{j+1} = w_j zeta_j,
    zeta_{j+1} = zeta_j rho).  Against the oracle and against the per-sample kernel (option signal_lin = 0)."""
    import torch
    rf = (np.array([0.0]), np.array([1e-4]), np.array([(np.pi / 2) / (W.GAMMA * 1e-4)]), np.array([0.0]))
    dwell = 4e-6
    t1 = 4e-4 + n_adc * dwell
    g = {0: ([2e-4, 3e-4, t1], [0, 1e-3, 1e-3]), 1: ([2e-4, 3e-4, t1], [0, -5e-4, -5e-4])}
    adc = 3.5e-4 + (np.arange(n_adc) + 0.5) * dwell
    s = seq(g=g, rf=rf, adc=adc, t_end=t1 + 1e-4, dt_rf_max=1.0)
    ph, v = moving_phantom(700, 31)
    out = {}
    for lin in ("1", "0"):
        out[lin], _ = run_both(B, oracle_mod, ph, s, v, 1e-5, f"motion recurrence {phase_mode} lin={lin}", phase_mode=phase_mode,
                               options={"signal_lin": int(lin)})
    emax, nrmse = errors(out["1"], out["0"])
    print(f"motion recurrence on/off {phase_mode}: max {emax:.3e} nrmse {nrmse:.3e}")
    assert 0 < emax <= 3e-5 and nrmse <= 8e-6


# ------------------------------------------------------------------------------------------------------------------
# General motion x(t) = x + a u(t) (BLOCH_MOTION_WAVEFORM; "motion field u(x, t)", reading M2)
# ------------------------------------------------------------------------------------------------------------------
def amplitudes(n, seed, scale=3e-3):
    rng = np.random.default_rng(seed)
    return tuple(rng.uniform(-scale, scale, n) for _ in range(3))


@pytest.mark.parametrize("phase_mode", ["fp32", "fp64"])
def test_epi_under_sinusoidal_nonrigid_displacement(B, oracle_mod, phase_mode):
    """Config-1-like EPI while every spin oscillates with its own amplitude vector (up to 3 mm) on a shared 200 Hz
    sinusoid given by 20 vertices per period: RF block, ramps, blips and plateaus all see the moving spins; the
    Cartesian-recurrence kernel must only take the groups on which the waveform is linear (the planner's parabola
    check), the rest goes through the per-sample kernel."""
    w = W.small("1")
    n = w.phantom.n
    wt = np.arange(int(w.seq.t_end / 2.5e-4) + 2) * 2.5e-4
    wf = (wt, np.sin(2 * np.pi * 200.0 * wt))
    a = amplitudes(n, 41)
    sig, ref = run_both(B, oracle_mod, w.phantom, w.seq, a, 2e-5, f"EPI sinusoidal motion {phase_mode}", phase_mode=phase_mode,
                        waveform=wf, max_speed_mps=6e-3)
    static = oracle_mod.simulate(w.phantom, w.seq)
    assert errors(ref, static)[0] > 1e-2, "the motion must change the signal for the test to mean anything"
    run_both(B, oracle_mod, w.phantom, w.seq, a, 2e-5, f"same through the host entry {phase_mode}", phase_mode=phase_mode,
             waveform=wf, host=True, max_speed_mps=6e-3)


def test_waveform_u_equal_t_is_bitwise_the_linear_motion_plan(B, oracle_mod):
    """u(t) = t as a two-vertex waveform builds the same tables as BLOCH_MOTION_LINEAR: signal and final state bitwise."""
    import torch
    w = W.small("3m")
    dev = B.phantom_to_device(w.phantom)
    vel = tuple(torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda() for a in w.velocity)
    out = []
    for kw in (dict(motion="linear"), dict(motion="waveform", waveform=([0.0, w.seq.t_end], [0.0, w.seq.t_end]))):
        plan = B.Plan(w.seq, phase_mode="fp64", dt_max=w.dt_max, **kw)
        Mxy = torch.zeros(w.phantom.n, 2, dtype=torch.float32, device="cuda")
        Mz = torch.zeros(w.phantom.n, dtype=torch.float32, device="cuda")
        sig = plan.simulate(*dev, Mxy=Mxy, Mz=Mz, velocity=vel)
        assert plan.status() == 0
        out.append((sig.cpu().numpy(), Mxy.cpu().numpy(), Mz.cpu().numpy()))
        plan.close()
    for a, b in zip(*out):
        assert np.array_equal(a.view(np.float32), b.view(np.float32))


def test_stop_and_go_motion_slice_selective_rf_and_per_spin_output(B, oracle_mod):
    """A displacement that ramps up during the slice-selective pulse, holds through the readout prephaser and returns
    during the readout (stop-and-go): motion RF tiles with a non-linear u, and per-spin output."""
    n_rf = 300
    dt = 1e-6
    tm = (np.arange(n_rf) + 0.5) * dt
    env = np.sinc(4.0 * (tm - n_rf * dt / 2) / (n_rf * dt))
    b1 = env * np.deg2rad(70) / (W.GAMMA * dt * env.sum())
    rf = (2e-4 + np.arange(n_rf) * dt, np.full(n_rf, dt), b1, np.zeros(n_rf))
    g = {2: ([1e-4, 2e-4, 5e-4, 6e-4, 8e-4, 9e-4], [0, 15e-3, 15e-3, 0, -11e-3, 0]),
         0: ([1.0e-3, 1.1e-3, 2.6e-3, 2.7e-3], [0, 7e-3, 7e-3, 0])}
    adc = 1.1e-3 + (np.arange(300) + 0.5) * 5e-6
    s = seq(g=g, rf=rf, adc=adc, t_end=3e-3, dt_rf_max=dt)
    wf = ([1.5e-4, 4.5e-4, 1.6e-3, 2.2e-3], [0.0, 1.0, 1.0, 0.0])
    ph, _ = moving_phantom(900, 43)
    a = amplitudes(ph.n, 44, scale=2e-3)
    run_both(B, oracle_mod, ph, s, a, 1e-5, "stop-and-go, slice-select", waveform=wf, max_speed_mps=4e-3)
    sub = ph.subset(np.arange(31))
    run_both(B, oracle_mod, sub, s, tuple(x[:31] for x in a), 1e-5, "stop-and-go, per spin", waveform=wf,
             output_mode="per_spin", max_speed_mps=4e-3)


def test_waveform_plan_argument_errors(B):
    s = W.small("1").seq
    for kw, code in ((dict(motion="waveform"), -1), (dict(motion="waveform", waveform=([1e-3, 5e-4], [0.0, 1.0])), -2),
                     (dict(motion="waveform", waveform=([0.0, 1e-3], [0.0, float("nan")])), -1)):
        with pytest.raises(B.BlochError) as e:
            B.Plan(s, **kw)
        assert e.value.code == code


def test_full_config3_under_periodic_nonrigid_motion(B, oracle_mod):
    """Workload 3w at full size (131,072 spins, EPI 128 x 128, fp64 phase, off-resonance, breathing-like non-rigid
    displacement), whole oracle."""
    import torch
    w = W.make("3w")
    plan = B.Plan(w.seq, **w.plan_kw)
    dev = B.phantom_to_device(w.phantom)
    amp = tuple(torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda() for a in w.velocity)
    Mxy = torch.zeros(w.phantom.n, 2, dtype=torch.float32, device="cuda")
    Mz = torch.zeros(w.phantom.n, dtype=torch.float32, device="cuda")
    sig = plan.simulate(*dev, Mxy=Mxy, Mz=Mz, velocity=amp)
    assert plan.status() == 0
    plan.close()
    ref, rxy, rz = oracle_mod.simulate(w.phantom, w.seq, velocity=w.velocity, dt_max=w.dt_max, waveform=w.waveform,
                                       return_state=True)
    m = Mxy.cpu().numpy()
    for name, got, want in (("signal", sig.cpu().numpy(), ref),
                            ("state", np.concatenate([m[:, 0] + 1j * m[:, 1], Mz.cpu().numpy().astype(np.complex128)]),
                             np.concatenate([rxy, rz.astype(np.complex128)]))):
        emax, nrmse = errors(got, want)
        print(f"config 3w full-size {name}: max {emax:.3e} nrmse {nrmse:.3e}")
        assert emax <= TOL_MAX and nrmse <= TOL_NRMSE
    static = oracle_mod.simulate(w.phantom.subset(np.arange(0, w.phantom.n, 64)), w.seq)
    moving = oracle_mod.simulate(w.phantom.subset(np.arange(0, w.phantom.n, 64)), w.seq,
                                 velocity=tuple(a[::64] for a in w.velocity), dt_max=w.dt_max, waveform=w.waveform)
    assert errors(moving, static)[0] > 1e-2
