"""Randomised GPU-vs-oracle parity (pytest -m gpu): seeded random sequences -- gradient vertices on all axes, several
RF bursts with random complex samples and step lengths, ADC samples scattered over the RF-free parts (including
on RF boundaries and at t = 0 / t_end), random phantoms and initial states; every output mode, both phase modes,
with and without motion.  Same acceptance as the other parity tests."""
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


def random_case(seed):
    rng = np.random.default_rng(1000 + seed)
    t_end = float(rng.uniform(4e-3, 12e-3))
    # RF bursts: disjoint windows, each with its own step length and random complex samples
    n_burst = int(rng.integers(1, 4))
    edges = np.sort(rng.uniform(0.05, 0.95, 2 * n_burst)) * t_end
    rf_t, rf_dt, rf_re, rf_im = [], [], [], []
    windows = []
    for k in range(n_burst):
        a, b = edges[2 * k], edges[2 * k + 1]
        dt = float(rng.choice([1e-6, 2e-6, 5e-6, 1e-5]))
        m = int(min(max(1, (b - a) // dt), 400))
        amp = rng.uniform(1e-6, 12e-6)
        rf_t.append(a + np.arange(m) * dt)
        rf_dt.append(np.full(m, dt))
        rf_re.append(amp * rng.uniform(-1, 1, m))
        rf_im.append(amp * rng.uniform(-1, 1, m))
        windows.append((a, a + m * dt))
    rf = tuple(np.concatenate(x) for x in (rf_t, rf_dt, rf_re, rf_im))
    # gradients: random vertices per axis
    g = {}
    for ax in range(3):
        nv = int(rng.integers(0, 9))
        if nv:
            g[ax] = (np.sort(rng.uniform(0, t_end, nv)), rng.uniform(-15e-3, 15e-3, nv))
    # ADC: random times outside the RF windows, plus the window edges and the sequence ends
    cand = rng.uniform(0, t_end, 400)
    keep = np.ones(cand.size, dtype=bool)
    for a, b in windows:
        keep &= (cand < a - 1e-9) | (cand > b + 1e-9)
    extra = [0.0, t_end] + [w[0] for w in windows] + [w[1] for w in windows]
    adc = np.unique(np.concatenate([cand[keep], extra]))
    adc = adc[np.concatenate([[True], np.diff(adc) > 1e-9])]
    if windows[0][0] < 1e-9:
        adc = adc[adc > 0.0]
    s = seq(g=g, rf=rf, adc=adc, t_end=t_end, dt_rf_max=float(rng.choice([1e-6, 3e-6, 1.0])))
    n = int(rng.integers(1, 700))
    ph = W._phantom(rng.uniform(-.12, .12, n), rng.uniform(-.12, .12, n), rng.uniform(-.05, .05, n),
                    rng.uniform(0, 1, n), rng.uniform(.2, 3, n), rng.uniform(.01, .2, n), rng.uniform(-400, 400, n))
    f32 = lambda a: np.asarray(a, dtype=np.float32).astype(np.float64)
    state = (f32(rng.normal(0, .4, n)) + 1j * f32(rng.normal(0, .4, n)), f32(rng.uniform(-1, 1, n)))
    vel = tuple(f32(rng.uniform(-.3, .3, n)) for _ in range(3))
    return s, ph, state, vel, rng


@pytest.mark.parametrize("seed", range(12))
def test_random_sequences(B, oracle_mod, seed):
    import torch
    s, ph, state, vel, rng = random_case(seed)
    n = ph.n
    mode = ["sum", "per_spin", "grouped"][seed % 3]
    phase = ["fp32", "fp64"][(seed // 3) % 2]
    moving = seed % 4 == 1 or seed % 4 == 2
    use_state = seed % 2 == 0
    gs = 1
    if mode == "grouped":
        gs = int(rng.choice([d for d in range(1, n + 1) if n % d == 0]))
    kw = dict(output_mode=mode, phase_mode=phase)
    okw = dict(output_mode=mode)
    if mode == "grouped":
        kw["group_size"] = gs
        okw["group_size"] = gs
    dt_max = 0.0
    if moving:
        dt_max = float(rng.choice([2e-5, 1e-4]))
        kw.update(motion="linear", dt_max=dt_max)
        okw.update(velocity=vel, dt_max=dt_max)
    plan = B.Plan(s, **kw)
    dev = B.phantom_to_device(ph)
    if use_state:
        Mxy = torch.view_as_real(torch.from_numpy(state[0].astype(np.complex64)).cuda()).contiguous()
        Mz = torch.from_numpy(state[1].astype(np.float32)).cuda()
    else:
        Mxy = torch.zeros(n, 2, dtype=torch.float32, device="cuda")
        Mz = torch.zeros(n, dtype=torch.float32, device="cuda")
    v_dev = tuple(torch.from_numpy(a.astype(np.float32)).cuda() for a in vel) if moving else None
    sig = plan.simulate(*dev, Mxy=Mxy, Mz=Mz, init_equilibrium=not use_state, velocity=v_dev)
    torch.cuda.synchronize()
    plan.close()
    ref, rxy, rz = oracle_mod.simulate(ph, s, state=state if use_state else None, return_state=True, **okw)
    m = Mxy.cpu().numpy()
    got_state = np.concatenate([m[:, 0] + 1j * m[:, 1], Mz.cpu().numpy().astype(np.complex128)])
    ref_state = np.concatenate([rxy, rz.astype(np.complex128)])
    for name, g, r in (("signal", sig.cpu().numpy(), ref), ("state", got_state, ref_state)):
        g = np.asarray(g, dtype=np.complex128)
        scale = max(np.abs(r).max(), 1e-30)
        d = np.abs(g - r)
        emax, nrmse = d.max() / scale, np.sqrt(np.mean(d ** 2)) / scale
        print(f"seed {seed} {mode} {phase} moving={moving} state={use_state} n={n} gs={gs} {name}: "
              f"max {emax:.3e} nrmse {nrmse:.3e}")
        assert g.shape == r.shape
        assert emax <= TOL_MAX and nrmse <= TOL_NRMSE


@pytest.mark.parametrize("seed", range(12, 24))
def test_random_sequences_whole_sequence_kernel_and_coils(B, oracle_mod, seed):
    """The same random sequences on the paths added later: the whole-sequence kernel (forced where the planner's
    phase choice is fp32, SUM_ALL; odd seeds from a supplied state) and multi-coil receive with 1-9 random smooth coil maps (per-block path, both
    phase modes)."""
    import torch
    s, ph, state, vel, rng = random_case(seed)
    n = ph.n
    use_state = seed % 2 == 1
    dev = B.phantom_to_device(ph)

    def fresh_state():
        if use_state:
            return (torch.view_as_real(torch.from_numpy(state[0].astype(np.complex64)).cuda()).contiguous(),
                    torch.from_numpy(state[1].astype(np.float32)).cuda())
        return (torch.zeros(n, 2, dtype=torch.float32, device="cuda"), torch.zeros(n, dtype=torch.float32, device="cuda"))

    def compare(what, g, r):
        g = np.asarray(g, dtype=np.complex128)
        scale = max(np.abs(r).max(), 1e-30)
        d = np.abs(g - r)
        emax, nrmse = d.max() / scale, np.sqrt(np.mean(d ** 2)) / scale
        print(f"seed {seed} n={n} {what}: max {emax:.3e} nrmse {nrmse:.3e}")
        assert g.shape == r.shape and emax <= TOL_MAX and nrmse <= TOL_NRMSE, what

    # (1) whole-sequence kernel
    ref, rxy, rz = oracle_mod.simulate(ph, s, state=state if use_state else None, return_state=True)
    ref_state = np.concatenate([rxy, rz.astype(np.complex128)])
    plan = B.Plan(s, path="fused")   # phase AUTO: 9 of the 12 sequences resolve to fp32, which the kernel needs
    if plan.info["phase_mode"] == B.PHASE_FP32 and B.bloch_plan_uses_fused(plan.handle, n):
        Mxy, Mz = fresh_state()
        sig = plan.simulate(*dev, Mxy=Mxy, Mz=Mz, init_equilibrium=not use_state)
        torch.cuda.synchronize()
        m = Mxy.cpu().numpy()
        compare("fused signal", sig.cpu().numpy(), ref)
        compare("fused state", np.concatenate([m[:, 0] + 1j * m[:, 1], Mz.cpu().numpy().astype(np.complex128)]), ref_state)
    plan.close()
    # (2) multi-coil receive
    n_coils = int(rng.integers(1, 10))
    cw = (rng.uniform(.2, 1, (n_coils, 1)) * np.exp(1j * (rng.uniform(-20, 20, (n_coils, 1)) * ph.x[None, :] +
                                                        rng.uniform(-20, 20, (n_coils, 1)) * ph.y[None, :])) /
          (1.0 + 30.0 * (ph.x[None, :] - rng.uniform(-.1, .1, (n_coils, 1))) ** 2)).astype(np.complex64)
    refc = oracle_mod.simulate(ph, s, state=state if use_state else None, coils=cw.astype(np.complex128))
    plan = B.Plan(s, phase_mode=["fp32", "fp64"][seed % 2])
    Mxy, Mz = fresh_state()
    sigc = plan.simulate(*dev, Mxy=Mxy, Mz=Mz, init_equilibrium=not use_state, coils=torch.from_numpy(cw).cuda())
    torch.cuda.synchronize()
    plan.close()
    compare(f"{n_coils} coils", sigc.cpu().numpy(), refc)
