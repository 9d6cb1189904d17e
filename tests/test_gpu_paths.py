"""GPU-vs-oracle parity on inputs chosen to drive every code path of the kernels (pytest -m gpu):
RF tiers 0/1/2, compact and general step tiles, tiles cut where the step length changes, the signal kernel's
series / per-sample exponential, P = 1, 2, 4 launch shapes with ragged tails, and batched second passes.
Same acceptance as test_gpu_parity.py."""
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
    scale = max(np.abs(ref).max(), 1e-300)
    d = np.abs(got - ref)
    return d.max() / scale, np.sqrt(np.mean(d ** 2)) / scale


def check(B, oracle_mod, ph, s, what, output_mode="sum", **plan_kw):
    """Both execution paths (one launch per block; the whole-sequence kernel where the plan qualifies) against
    the oracle.  Returns the launch count of the per-block path."""
    import torch
    ref, rxy, rz = oracle_mod.simulate(ph, s, output_mode=output_mode, return_state=True)
    ref_state = np.concatenate([rxy, rz.astype(np.complex128)])
    dev = B.phantom_to_device(ph)
    launches = None
    for path in ("per_block", "fused"):
        plan = B.Plan(s, path=path, output_mode=output_mode, **plan_kw)
        if path == "fused" and not B.bloch_plan_uses_fused(plan.handle, ph.n):
            plan.close()
            continue
        Mxy = torch.zeros(ph.n, 2, dtype=torch.float32, device="cuda")
        Mz = torch.zeros(ph.n, dtype=torch.float32, device="cuda")
        sig = plan.simulate(*dev, Mxy=Mxy, Mz=Mz)
        torch.cuda.synchronize()
        if path == "per_block":
            launches = B.bloch_plan_last_launches(plan.handle)
        plan.close()
        m = Mxy.cpu().numpy()
        got_state = np.concatenate([m[:, 0] + 1j * m[:, 1], Mz.cpu().numpy().astype(np.complex128)])
        for name, g, r in (("signal", sig.cpu().numpy(), ref), ("state", got_state, ref_state)):
            if r.size == 0:
                continue
            emax, nrmse = errors(g, r)
            print(f"{what} [{path}] {name}: max {emax:.3e} nrmse {nrmse:.3e}")
            assert emax <= TOL_MAX and nrmse <= TOL_NRMSE, f"{what} [{path}] {name}: max {emax:.3e} nrmse {nrmse:.3e}"
    return launches


def rand_phantom(n, seed, zmax=0.01, dwmax=300.0, t2=(0.03, 0.3)):
    rng = np.random.default_rng(seed)
    return W._phantom(rng.uniform(-.1, .1, n), rng.uniform(-.1, .1, n), rng.uniform(-zmax, zmax, n),
                      rng.uniform(.5, 1, n), rng.uniform(.3, 2, n), rng.uniform(*t2, n), rng.uniform(-dwmax, dwmax, n))


def sinc_rf(t0, dur, n, flip):
    dt = dur / n
    tm = (np.arange(n) + 0.5) * dt
    env = np.sinc(4.0 * (tm - dur / 2) / dur)
    b1 = env * flip / (W.GAMMA * dt * env.sum())
    return t0 + np.arange(n) * dt, np.full(n, dt), b1, np.zeros(n)


@pytest.mark.parametrize("dt_rf,zmax,tier", [(1e-6, 0.002, 0), (1e-6, 0.08, 1), (4e-6, 0.08, 2)])
def test_rf_tiers_on_a_slice_select_plateau(B, oracle_mod, dt_rf, zmax, tier):
    """|w|^2 per step is set by gamma*G*z*dt: 10 mT/m, z up to 2 mm / 8 cm, dt 1 / 4 us -> tiers 0 / 1 / 2."""
    n_rf = int(round(1e-3 / dt_rf))
    rf = sinc_rf(2e-4, 1e-3, n_rf, np.deg2rad(40))
    g = {2: ([1e-4, 2e-4, 1.2e-3, 1.3e-3, 1.8e-3, 1.9e-3], [0, 10e-3, 10e-3, 0, -8e-3, 0]),
         0: ([1.4e-3, 1.5e-3, 2.5e-3, 2.6e-3], [0, 5e-3, 5e-3, 0])}
    adc = 1.5e-3 + (np.arange(300) + 0.5) * 3e-6
    s = seq(g=g, rf=rf, adc=adc, t_end=3e-3, dt_rf_max=dt_rf)
    ph = rand_phantom(777, 100 + tier, zmax=zmax)
    wz = W.GAMMA * 10e-3 * zmax * dt_rf
    assert (wz * wz <= 2 ** -8) == (tier == 0) and (wz * wz > 0.25) == (tier == 2)
    check(B, oracle_mod, ph, s, f"RF tier {tier}")


def test_rf_on_gradient_ramps_and_changing_step_length(B, oracle_mod):
    """General (32-B) step records: the gradient changes from step to step; RF samples of three different
    lengths force tile cuts where dt changes; 300 steps of one dt span more than one 128-step tile."""
    dts = np.concatenate([np.full(300, 1e-6), np.full(40, 5e-6), np.full(7, 2e-6), np.full(150, 1e-6)])
    t0 = 1e-4 + np.concatenate([[0.0], np.cumsum(dts)[:-1]])
    rng = np.random.default_rng(5)
    b1 = rng.uniform(-4e-6, 4e-6, dts.size)
    b1i = rng.uniform(-4e-6, 4e-6, dts.size)
    t_rf_end = t0[-1] + dts[-1]
    g = {0: ([0.0, 3e-4, 5e-4, 9e-4], [0, 12e-3, -6e-3, 0]),
         1: ([5e-5, 4e-4, 1.5e-3], [0, 8e-3, 0]),
         2: ([0.0, 2e-4, 6e-4, 1.2e-3], [3e-3, 3e-3, -9e-3, 0])}
    adc = t_rf_end + 1e-5 + np.arange(77) * 7e-6
    s = seq(g=g, rf=(t0, dts, b1, b1i), adc=adc, t_end=2.5e-3, dt_rf_max=1.0)
    check(B, oracle_mod, rand_phantom(333, 6), s, "RF on ramps, mixed dt")


@pytest.mark.parametrize("n_adc", [1, 5, 40, 100, 200, 300, 700, 1023, 2049, 2300])
def test_signal_launch_shapes_and_ragged_tails(B, oracle_mod, n_adc):
    """n_adc selects the CTA size (32 ... 256 threads below 256 points), P = 1 (< 512 points), 2 (< 1024), 4 (< 2048) or 8
    and leaves ragged point tiles; 1111 spins leave a
    ragged spin tile."""
    rf = (np.array([0.0]), np.array([1e-4]), np.array([(np.pi / 3) / (W.GAMMA * 1e-4)]), np.array([0.0]))
    g = {0: ([2e-4, 3e-4, 9e-3], [0, 4e-3, 4e-3]), 1: ([2e-4, 3e-4, 9e-3], [0, -2e-3, 1e-3])}
    adc = 3.5e-4 + (np.arange(n_adc) + 0.5) * 4e-6
    s = seq(g=g, rf=rf, adc=adc, t_end=1e-2, dt_rf_max=1.0)
    check(B, oracle_mod, rand_phantom(1111, 7), s, f"signal n_adc={n_adc}")


def test_signal_series_fallback_when_adjacent_samples_are_far_apart(B, oracle_mod):
    """Bursts of 5 samples separated by 1.5 ms with T2 down to 5 ms: (tau_j - tau_0)/T2 reaches 0.3 inside a
    thread's 4 adjacent points, so those warps must take one MUFU.EX2 per sample; others keep the series."""
    rf = (np.array([0.0]), np.array([1e-4]), np.array([(np.pi / 2) / (W.GAMMA * 1e-4)]), np.array([0.0]))
    bursts = 2e-4 + np.arange(300)[:, None] * 1.5e-3 + np.arange(5)[None, :] * 5e-6
    adc = np.sort(bursts.ravel())
    g = {0: ([1.5e-4, 2e-4, adc[-1] + 1e-4], [0, 1e-3, 1e-3])}
    s = seq(g=g, rf=rf, adc=adc, t_end=adc[-1] + 2e-4, dt_rf_max=1.0)
    check(B, oracle_mod, rand_phantom(600, 8, t2=(0.005, 0.05)), s, "series fallback")


def test_batched_second_pass_over_many_blocks(B, oracle_mod):
    """20 TRs with one readout each: the precession blocks share partial-sum batches; forcing tiny blocks
    (max_block_points) multiplies the number of blocks per batch."""
    w = W.small("5")
    a = check(B, oracle_mod, w.phantom, w.seq, "batched reduce")
    b = check(B, oracle_mod, w.phantom, w.seq, "batched reduce, cut blocks", max_block_points=50)
    assert b > a


def test_adiabatic_inversion_recovery_long_soft_pulse(B, oracle_mod):
    """The paper's stated weak spot: a long soft pulse with a frequency sweep.  10.24 ms hyperbolic-
    secant inversion (10,240 steps of phase-modulated complex B1 = 80 step tiles) under a slice gradient, spins spread
    over +-1.5 kHz of off-resonance so that some lie inside, some on the edge of and some outside the inverted band,
    then inversion recovery, a hard 90 and a gradient-echo readout."""
    mu, beta, T, n = 5.0, 800.0, 10.24e-3, 10240
    dt = T / n
    tm = (np.arange(n) + 0.5) * dt - T / 2
    amp = 4500.0 / W.GAMMA / np.cosh(beta * tm)
    phi = mu * np.log(1.0 / np.cosh(beta * tm))
    t90 = 40e-3
    b90 = (np.pi / 2) / (W.GAMMA * 1e-4)
    rf = (np.concatenate([1e-4 + np.arange(n) * dt, t90 + np.arange(10) * 1e-5]),
          np.concatenate([np.full(n, dt), np.full(10, 1e-5)]),
          np.concatenate([amp * np.cos(phi), np.full(10, b90)]),
          np.concatenate([amp * np.sin(phi), np.zeros(10)]))
    g = {2: ([0.0, 1e-4, 1e-4 + T, 2e-4 + T], [0, 2e-3, 2e-3, 0]),
         0: ([t90 + 2e-4, t90 + 3e-4, t90 + 8e-4, t90 + 9e-4, t90 + 2.0e-3, t90 + 2.1e-3], [0, -6e-3, -6e-3, 6e-3, 6e-3, 0])}
    adc = t90 + 9.5e-4 + (np.arange(256) + 0.5) * 4e-6
    s = seq(g=g, rf=rf, adc=adc, t_end=t90 + 3e-3, dt_rf_max=1.0)
    ph = rand_phantom(3000, 21, zmax=0.01, dwmax=2 * np.pi * 1500.0, t2=(0.03, 0.3))
    check(B, oracle_mod, ph, s, "adiabatic inversion recovery")
    _, _, rz = oracle_mod.simulate(ph, seq(g={2: g[2]}, rf=tuple(a[:n] for a in rf), t_end=2e-4 + T, dt_rf_max=1.0),
                                   return_state=True)
    frac = rz / ph.M0
    assert (frac < -0.8).sum() > 300 and (frac > 0.8).sum() > 300, "the phantom must straddle the inverted band"


def test_off_centre_slices_by_rf_phase_ramps(B, oracle_mod):
    """Two slice-selective pulses with frequency offsets of +3 kHz and -2 kHz (phase ramps on the complex B1: the step
    records change in both components from step to step), each followed by a readout; spins across 4 cm of z."""
    T, n, Gz = 2e-3, 2000, 8e-3
    dt = T / n
    tm = (np.arange(n) + 0.5) * dt
    env = np.sinc(4.0 * (tm - T / 2) / T)
    b1 = env * (np.pi / 4) / (W.GAMMA * dt * env.sum())
    parts, g2, adc = [], [[], []], []
    gx = [[], []]
    for k, df in enumerate((3000.0, -2000.0)):
        t0 = 1e-4 + k * 6e-3
        ph = -2 * np.pi * df * tm
        parts.append((t0 + np.arange(n) * dt, np.full(n, dt), b1 * np.cos(ph), b1 * np.sin(ph)))
        g2[0] += [t0 - 1e-4, t0, t0 + T, t0 + T + 1e-4, t0 + T + 6e-4, t0 + T + 7e-4]
        g2[1] += [0.0, Gz, Gz, -Gz, -Gz, 0.0]           # slice select, then a rephaser lobe
        gx[0] += [t0 + T + 8e-4, t0 + T + 9e-4, t0 + T + 2.9e-3, t0 + T + 3e-3]
        gx[1] += [0.0, 5e-3, 5e-3, 0.0]
        adc.append(t0 + T + 1e-3 + (np.arange(150) + 0.5) * 1e-5)
    rf = tuple(np.concatenate([p[i] for p in parts]) for i in range(4))
    s = seq(g={2: (g2[0], g2[1]), 0: (gx[0], gx[1])}, rf=rf, adc=np.concatenate(adc), t_end=13e-3, dt_rf_max=1.0)
    ph = rand_phantom(4000, 31, zmax=0.02, dwmax=100.0)
    check(B, oracle_mod, ph, s, "off-centre slices")


@pytest.mark.parametrize("jitter", [0.0, 2e-9, 3e-7])
def test_signal_decay_modes_equal_spacing_and_jitter(B, oracle_mod, jitter):
    """Equally spaced samples take the geometric decay (sample j = sample j-1 times exp(-dwell/T2)); samples jittered
    by a few ns still do (below the 1e-6 bound on |deviation|/T2 with T2 >= 5 ms), by 0.3 us fall back to the
    per-sample series.  4100 samples = P = 8 per thread with a ragged tail; short T2 makes the decay matter."""
    rng = np.random.default_rng(12)
    rf = (np.array([0.0]), np.array([1e-4]), np.array([(np.pi / 2) / (W.GAMMA * 1e-4)]), np.array([0.0]))
    adc = 3e-4 + (np.arange(4100) + 0.5) * 2e-6 + rng.uniform(-jitter, jitter, 4100)
    g = {0: ([2e-4, 3e-4, 9e-3], [0, 4e-3, 4e-3]), 1: ([2e-4, 3e-4, 9e-3], [0, -2e-3, 1e-3])}
    s = seq(g=g, rf=rf, adc=np.sort(adc), t_end=1e-2, dt_rf_max=1.0)
    check(B, oracle_mod, rand_phantom(900, 13, t2=(0.005, 0.05)), s, f"decay modes, jitter {jitter}")


@pytest.mark.parametrize("phase_mode", ["fp32", "fp64"])
def test_signal_rotation_recurrence_on_cartesian_lines(B, oracle_mod, phase_mode):
    """EPI-like train sampled THROUGH the ramps: the warps whose 8 (or 4) adjacent samples sit on a plateau take the
    rotation recurrence (k' advances by a constant step), those that touch a ramp or a blip must not.  Both against the
    oracle, and against the same kernel with the recurrence switched off (option signal_lin = 0)."""
    import torch
    rf = (np.array([0.0]), np.array([1e-4]), np.array([(np.pi / 2) / (W.GAMMA * 1e-4)]), np.array([0.0]))
    n_lines, flat, ramp, G = 12, 1.2e-3, 1.0e-4, 9e-3
    t, v, ty, vy = [2e-4], [0.0], [2e-4], [0.0]
    for ln in range(n_lines):
        sgn = 1.0 if ln % 2 == 0 else -1.0
        t0 = t[-1]
        t += [t0 + ramp, t0 + ramp + flat, t0 + 2 * ramp + flat]
        v += [sgn * G, sgn * G, 0.0]
        ty += [t0 + 2 * ramp + flat - 5e-5, t0 + 2 * ramp + flat - 2.5e-5, t0 + 2 * ramp + flat]
        vy += [0.0, 2e-3, 0.0]
    t_end = t[-1] + 1e-4
    adc = 2.1e-4 + (np.arange(int((t[-1] - 2.2e-4) / 4e-6)) + 0.5) * 4e-6   # ~4200 samples: P = 8, ragged tail
    s = seq(g={0: (t, v), 1: (ty, vy)}, rf=rf, adc=adc, t_end=t_end, dt_rf_max=1.0)
    ph = rand_phantom(1500, 21)
    check(B, oracle_mod, ph, s, f"recurrence {phase_mode}", phase_mode=phase_mode)
    dev = B.phantom_to_device(ph)
    out = {}
    for lin in ("1", "0"):
        plan = B.Plan(s, path="per_block", phase_mode=phase_mode, options={"signal_lin": int(lin)})
        out[lin] = plan.simulate(*dev).cpu().numpy()
        torch.cuda.synchronize()
        plan.close()
    emax, nrmse = errors(out["1"], out["0"])
    print(f"recurrence on/off {phase_mode}: max {emax:.3e} nrmse {nrmse:.3e}")
    assert 0 < emax <= 2e-5 and nrmse <= 5e-6      # different arithmetic (not bitwise), same answer


@pytest.mark.parametrize("phase_mode,n_adc", [("fp32", 2048), ("fp32", 4103), ("fp64", 2061), ("fp64", 8192)])
def test_signal_lin_kernel_on_all_cartesian_blocks(B, oracle_mod, phase_mode, n_adc):
    """A block of >= 2048 equally spaced samples on a plateau: the planner hands its first n - n % 16 samples to
    signal_lin_kernel (16 samples per thread, recurrence only) and the tail to signal_kernel<1>.  Against the oracle
    and against the per-sample kernel (option signal_lin = 0); short T2 (dwell / T2 up to 0.04) also drives the
    MUFU.EX2 form of q in the fp64 cases."""
    import torch
    rf = (np.array([0.0]), np.array([1e-4]), np.array([(np.pi / 2) / (W.GAMMA * 1e-4)]), np.array([0.0]))
    dwell = 4e-6 if phase_mode == "fp32" else 2e-4
    t1 = 4e-4 + n_adc * dwell
    g = {0: ([2e-4, 3e-4, t1], [0, 1e-3, 1e-3] if phase_mode == "fp32" else [0, 1e-4, 1e-4]),
         1: ([2e-4, 3e-4, t1], [0, -5e-4, -5e-4] if phase_mode == "fp32" else [0, -5e-5, -5e-5])}
    adc = 3.5e-4 + (np.arange(n_adc) + 0.5) * dwell
    s = seq(g=g, rf=rf, adc=adc, t_end=t1 + 1e-4, dt_rf_max=1.0)
    ph = rand_phantom(777, 23, t2=(0.03, 0.3) if phase_mode == "fp32" else (0.005, 0.3))
    launches = check(B, oracle_mod, ph, s, f"lin kernel {phase_mode} n_adc={n_adc}", phase_mode=phase_mode)
    pl = B.Plan(s, path="per_block", phase_mode=phase_mode)
    assert launches == B.bloch_plan_get_info(pl.handle)["n_launches"]      # the tail launch is counted by the planner
    pl.close()
    dev = B.phantom_to_device(ph)
    out = {}
    for lin in ("1", "0"):
        plan = B.Plan(s, path="per_block", phase_mode=phase_mode, options={"signal_lin": int(lin)})
        out[lin] = plan.simulate(*dev).cpu().numpy()
        torch.cuda.synchronize()
        plan.close()
    emax, nrmse = errors(out["1"], out["0"])
    print(f"lin kernel on/off {phase_mode} n_adc={n_adc}: max {emax:.3e} nrmse {nrmse:.3e}")
    assert 0 < emax <= 3e-5 and nrmse <= 8e-6     # fp32: both sit on the fp32 phase floor (no echo in this sequence)


@pytest.mark.parametrize("phase_mode", ["fp32", "fp64"])
def test_signal_lin_kernel_on_an_epi_train_of_short_lines(B, oracle_mod, phase_mode):
    """50 EPI lines of 48 samples on the plateaus only (ramps and blips between lines are not sampled): every aligned
    group of 16 lies inside one line, so the whole 2400-sample block goes to signal_lin_kernel although k' and tau
    jump between groups.  A second sequence shifts the first line by 5 samples: groups then straddle the line ends,
    the planner must NOT flag the block, and the per-warp choice inside signal_kernel takes over."""
    import torch
    rf = (np.array([0.0]), np.array([1e-4]), np.array([(np.pi / 2) / (W.GAMMA * 1e-4)]), np.array([0.0]))
    dwell, n_line, n_lines, ramp, G = 5e-6, 48, 50, 1e-4, 6e-3
    ph = rand_phantom(900, 29)
    dev = B.phantom_to_device(ph)
    for extra in (0, 5):
        t, v, ty, vy, adc = [2e-4], [0.0], [2e-4], [0.0], []
        for ln in range(n_lines):
            sgn = 1.0 if ln % 2 == 0 else -1.0
            t0 = t[-1]
            n_here = n_line + (extra if ln == 0 else 0)
            flat = n_here * dwell
            t += [t0 + ramp, t0 + ramp + flat, t0 + 2 * ramp + flat]
            v += [sgn * G, sgn * G, 0.0]
            adc.append(t0 + ramp + (np.arange(n_here) + 0.5) * dwell)
            ty += [t0 + 2 * ramp + flat - 5e-5, t0 + 2 * ramp + flat - 2.5e-5, t0 + 2 * ramp + flat]
            vy += [0.0, 1.5e-3, 0.0]
        adc = np.concatenate(adc)
        s = seq(g={0: (t, v), 1: (ty, vy)}, rf=rf, adc=adc, t_end=t[-1] + 1e-4, dt_rf_max=1.0)
        check(B, oracle_mod, ph, s, f"EPI short lines {phase_mode} shift={extra}", phase_mode=phase_mode)
        out = {}
        for lin in ("1", "0"):
            plan = B.Plan(s, path="per_block", phase_mode=phase_mode, options={"signal_lin": int(lin)})
            out[lin] = plan.simulate(*dev).cpu().numpy()
            torch.cuda.synchronize()
            plan.close()
        emax, nrmse = errors(out["1"], out["0"])
        print(f"EPI short lines on/off {phase_mode} shift={extra}: max {emax:.3e} nrmse {nrmse:.3e}")
        assert emax <= 3e-5 and nrmse <= 8e-6
        if extra == 0:
            assert emax > 0      # the recurrence kernel did run


@pytest.mark.parametrize("name", ["1", "2", "4", "5"])
def test_two_spins_per_thread_rf_kernel_is_bitwise_the_one_spin_kernel(B, oracle_mod, name):
    """rf_pair_kernel (BLOCH_OPT_RF_SPINS = 2): thread t owns spins t and t + ceil(n / 2) and shares the step record
    between them; every spin's own arithmetic is unchanged, so signal and final magnetisation are bitwise those of
    rf_kernel (odd spin counts, compact and general tiles, propagate at block starts), and match the oracle."""
    from test_gpu_parity import run_gpu
    w = W.small(name)
    out = {}
    for spins in (1, 2):
        out[spins] = run_gpu(B, w, want_state=True, path="per_block", options={"rf_spins": spins})
    for a, b in zip(out[1], out[2]):
        assert np.array_equal(np.asarray(a).view(np.float32), np.asarray(b).view(np.float32))
    ref, rxy, rz = oracle_mod.simulate(w.phantom, w.seq, output_mode=w.output_mode, return_state=True)
    emax, nrmse = errors(out[2][0], ref)
    assert emax <= 1e-4 and nrmse <= 1e-5
    # an odd number of spins: the last thread's second spin does not exist
    ph = w.phantom.subset(np.arange(w.phantom.n - (1 - w.phantom.n % 2)))
    assert ph.n % 2 == 1
    w2 = W.Workload(w.name, ph, w.seq, phase_mode=w.phase_mode, output_mode=w.output_mode)
    a = run_gpu(B, w2, want_state=True, path="per_block", options={"rf_spins": 1})
    b = run_gpu(B, w2, want_state=True, path="per_block", options={"rf_spins": 2})
    for u, v in zip(a, b):
        assert np.array_equal(np.asarray(u).view(np.float32), np.asarray(v).view(np.float32))


@pytest.mark.parametrize("path", ["per_block", "fused"])
def test_adc_samples_during_an_rf_pulse(B, oracle_mod, path):
    """ADC samples strictly inside an RF run, at its first and at its last instant (reading G7: Mxy after the step that
    ends at the sample's time): served through empty precession blocks that cut the run; signal and final state against
    the oracle, which integrates straight through."""
    from test_gpu_parity import run_gpu
    n_rf, dt = 600, 2e-6
    tm = (np.arange(n_rf) + 0.5) * dt
    env = np.sinc(4.0 * (tm - n_rf * dt / 2) / (n_rf * dt))
    b1 = env * np.deg2rad(80) / (W.GAMMA * dt * env.sum())
    rf = (np.arange(n_rf) * dt, np.full(n_rf, dt), b1 * np.cos(0.3), b1 * np.sin(0.3))
    t_rf = n_rf * dt
    g = {2: ([0.0, t_rf, t_rf + 1e-4, t_rf + 3e-4, t_rf + 4e-4], [8e-3, 8e-3, 0.0, -6e-3, 0.0]),
         0: ([t_rf + 4e-4, t_rf + 5e-4, t_rf + 1.5e-3], [0.0, 5e-3, 5e-3])}
    adc = np.concatenate([[0.0], np.arange(1, 30) * 20 * dt, [t_rf - 3e-6 + 1e-6], [t_rf],
                          t_rf + 5e-4 + np.arange(100) * 1e-5])
    s = seq(g=g, rf=rf, adc=adc, t_end=t_rf + 1.5e-3, dt_rf_max=dt)
    rng = np.random.default_rng(61)
    n = 1111
    ph = W._phantom(rng.uniform(-.08, .08, n), rng.uniform(-.08, .08, n), rng.uniform(-.004, .004, n),
                    rng.uniform(.5, 1, n), rng.uniform(.3, 2, n), rng.uniform(.03, .3, n), rng.uniform(-200, 200, n))
    w = W.Workload("adc_in_rf", ph, s, phase_mode="fp32")
    got, gxy, gz = run_gpu(B, w, want_state=True, path=path)
    ref, rxy, rz = oracle_mod.simulate(ph, s, return_state=True)
    assert np.abs(ref[1:31]).max() > 0.05 * np.abs(ref).max()      # the in-pulse samples carry signal
    emax, nrmse = errors(got, ref)
    print(f"ADC inside RF, {path}: max {emax:.3e} nrmse {nrmse:.3e}")
    assert emax <= 1e-4 and nrmse <= 1e-5
    emax, nrmse = errors(np.concatenate([gxy, gz.astype(np.complex128)]), np.concatenate([rxy, rz.astype(np.complex128)]))
    assert emax <= 1e-4 and nrmse <= 1e-5


@pytest.mark.parametrize("name", ["1", "2", "4", "5"])
def test_rf_const_kernel_is_bitwise_the_tile_kernel(B, oracle_mod, name):
    """rf_const_kernel (BLOCH_OPT_RF_CONST, the default for static plans whose RF tiles are compact): the step records
    are passed by value as kernel parameters and reach the FMAs as uniform operands; the arithmetic is rf_kernel's,
    operation for operation, so signal and final magnetisation are bitwise equal (and match the oracle)."""
    from test_gpu_parity import run_gpu
    w = W.small(name)
    out = {c: run_gpu(B, w, want_state=True, path="per_block", phase_mode="fp32", options={"rf_const": c}) for c in (0, 2)}
    for a, b in zip(out[0], out[2]):
        assert np.array_equal(np.asarray(a).view(np.float32), np.asarray(b).view(np.float32))
    ref = oracle_mod.simulate(w.phantom, w.seq, output_mode=w.output_mode)
    emax, nrmse = errors(out[2][0], ref)
    assert emax <= 1e-4 and nrmse <= 1e-5


def test_rf_const_kernel_limits_and_fallback(B, oracle_mod):
    """A 2000-step pulse on a slice-select plateau is 16 compact tiles = one parameter block: rf_const_kernel.  A
    5000-step pulse does not fit one block (2000 steps) and a pulse that runs over the gradient ramps has general
    (32-B) records: both keep rf_kernel.  All against the oracle, and bitwise against the tile kernel."""
    import torch
    g_plateau = {2: ([1e-4, 2e-4, 5.4e-3, 5.5e-3, 5.9e-3, 6.0e-3], [0, 6e-3, 6e-3, 0, -7e-3, 0]),
                 0: ([6.1e-3, 6.2e-3, 7.2e-3, 7.3e-3], [0, 5e-3, 5e-3, 0])}
    g_ramps = {2: ([1e-4, 2.5e-3, 5.4e-3, 5.5e-3, 5.9e-3, 6.0e-3], [0, 6e-3, 2e-3, 0, -7e-3, 0]), 0: g_plateau[0]}
    adc = 6.2e-3 + (np.arange(200) + 0.5) * 4e-6
    ph = rand_phantom(1111, 42, zmax=0.004)
    for n_rf, g, kernel in ((2000, g_plateau, "rf_const_kernel"), (5000, g_plateau, "rf_kernel<0>"),
                            (2000, g_ramps, "rf_kernel<0>")):
        rf = sinc_rf(3e-4, n_rf * 1e-6, n_rf, np.deg2rad(60))
        s = seq(g=g, rf=rf, adc=adc, t_end=8e-3, dt_rf_max=1e-6)
        ref = oracle_mod.simulate(ph, s)
        res = {}
        for c in (2, 0):   # 2: rf_const_kernel where it applies whatever the number of spins (1: from 16,384 spins on)
            plan = B.Plan(s, path="per_block", phase_mode="fp32", options={"rf_const": c})
            Mxy = torch.zeros(ph.n, 2, device="cuda")
            Mz = torch.zeros(ph.n, device="cuda")
            sig = plan.simulate(*B.phantom_to_device(ph), Mxy=Mxy, Mz=Mz)
            torch.cuda.synchronize()
            res[c] = (sig.cpu().numpy(), Mxy.cpu().numpy(), Mz.cpu().numpy())
            name = B.bloch_plan_last_kernel(plan.handle, "rf")["name"]
            assert name == (kernel if c else "rf_kernel<0>"), (n_rf, name)
            assert B.bloch_plan_last_launches(plan.handle) == plan.info["n_launches"]
            plan.close()
        for a, b in zip(res[0], res[2]):
            assert np.array_equal(a.view(np.float32), b.view(np.float32))
        emax, nrmse = errors(res[2][0], ref)
        print(f"{n_rf}-step pulse ({kernel}): max {emax:.3e} nrmse {nrmse:.3e}")
        assert emax <= TOL_MAX and nrmse <= TOL_NRMSE
    plan = B.Plan(s, path="per_block", phase_mode="fp32")          # default (1): 1111 spins are below the threshold
    plan.simulate(*B.phantom_to_device(ph))
    torch.cuda.synchronize()
    assert B.bloch_plan_last_kernel(plan.handle, "rf")["name"] == "rf_kernel<0>"
    plan.close()
