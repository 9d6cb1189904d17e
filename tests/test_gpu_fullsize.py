"""GPU-vs-oracle parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(run on the B200 box: pytest -m gpu).

Configs 1-3 are small enough for the oracle to run whole.  For configs 4 and 5 (1e11 spin*steps, hours of
oracle time) the check is split into pieces that together fix the full-size result:
  (a) per-spin outputs the oracle can compute one by one: the final magnetisation of sampled spins, taken from
      the full-size run, against the oracle on exactly those spins;
  (b) the summed signal of an evenly spaced spin subset against the oracle on that subset (same plan, same
      kernels, same time tiles);
  (c) superposition (invariant I3): S(full) = S(subset) + S(complement) to fp32 rounding, which ties the full-size
      launch shape (spin chunks, partial sums, second pass) to (b).
Dictionary mode 5b (PER_SPIN) is checked on sampled rows of the full 100,000 x 1000 output.
"""
import numpy as np
import pytest

from paper_2301_02702_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_MAX = 1e-4      # BASELINE.json north_star
TOL_NRMSE = 1e-5    # reading G17


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


def assert_parity(got, ref, what):
    emax, nrmse = errors(got, ref)
    print(f"{what}: max {emax:.3e} nrmse {nrmse:.3e}")
    assert emax <= TOL_MAX and nrmse <= TOL_NRMSE, f"{what}: max {emax:.3e} nrmse {nrmse:.3e}"


def gpu_run(B, plan, ph, want_state=False):
    import torch
    dev = B.phantom_to_device(ph)
    Mxy = Mz = None
    if want_state:
        Mxy = torch.zeros(ph.n, 2, dtype=torch.float32, device="cuda")
        Mz = torch.zeros(ph.n, dtype=torch.float32, device="cuda")
    sig = plan.simulate(*dev, Mxy=Mxy, Mz=Mz)
    torch.cuda.synchronize()
    if want_state:
        m = Mxy.cpu().numpy()
        return sig.cpu().numpy(), m[:, 0] + 1j * m[:, 1], Mz.cpu().numpy()
    return sig.cpu().numpy()


def state_vec(mxy, mz):
    return np.concatenate([np.asarray(mxy, dtype=np.complex128), np.asarray(mz, dtype=np.complex128)])


@pytest.mark.parametrize("name", ["1", "2", "3"])
def test_full_config_against_whole_oracle(B, oracle_mod, name):
    w = W.make(name)
    plan = B.Plan(w.seq, phase_mode=w.phase_mode, output_mode=w.output_mode)
    got, gxy, gz = gpu_run(B, plan, w.phantom, want_state=True)
    plan.close()
    ref, rxy, rz = oracle_mod.simulate(w.phantom, w.seq, return_state=True)
    assert_parity(got, ref, f"config {name} full-size signal")
    assert_parity(state_vec(gxy, gz), state_vec(rxy, rz), f"config {name} full-size final state")


@pytest.mark.parametrize("name,n_sub,n_state", [("4", 1024, 64), ("5", 128, 32)])
def test_large_config_by_samples_subset_and_superposition(B, oracle_mod, name, n_sub, n_state):
    w = W.make(name)
    n = w.phantom.n
    plan = B.Plan(w.seq, phase_mode=w.phase_mode, output_mode=w.output_mode)
    full, gxy, gz = gpu_run(B, plan, w.phantom, want_state=True)
    again = gpu_run(B, plan, w.phantom)
    assert np.array_equal(full.view(np.float32), again.view(np.float32)), "full-size run not bitwise reproducible"
    # (a) sampled spins' final magnetisation from the full-size run
    rng = np.random.default_rng(11)
    idx = np.sort(rng.choice(n, n_state, replace=False))
    _, rxy, rz = oracle_mod.simulate(w.phantom.subset(idx), w.seq, return_state=True)
    assert_parity(state_vec(gxy[idx], gz[idx]), state_vec(rxy, rz), f"config {name} sampled final state")
    # (b) evenly spaced subset against the oracle
    sub = np.linspace(0, n - 1, n_sub).astype(np.int64)
    mask = np.ones(n, dtype=bool)
    mask[sub] = False
    s_sub = gpu_run(B, plan, w.phantom.subset(sub))
    ref_sub = oracle_mod.simulate(w.phantom.subset(sub), w.seq)
    assert_parity(s_sub, ref_sub, f"config {name} subset signal ({n_sub} spins)")
    # (c) superposition ties the full-size launch to (b)
    s_rest = gpu_run(B, plan, w.phantom.subset(np.flatnonzero(mask)))
    plan.close()
    emax, nrmse = errors(s_sub.astype(np.complex128) + s_rest, full)
    print(f"config {name} superposition: max {emax:.3e} nrmse {nrmse:.3e}")
    assert emax < 5e-6 and nrmse < 1e-6


def test_dictionary_full_size_sampled_rows(B, oracle_mod):
    w = W.make("5b")
    plan = B.Plan(w.seq, phase_mode=w.phase_mode, output_mode=w.output_mode)
    import torch
    dev = B.phantom_to_device(w.phantom)
    sig = plan.simulate(*dev)
    torch.cuda.synchronize()
    assert tuple(sig.shape) == (w.phantom.n, plan.info["n_adc"])
    rng = np.random.default_rng(12)
    idx = np.sort(rng.choice(w.phantom.n, 48, replace=False))
    rows = sig[torch.from_numpy(idx).cuda()].cpu().numpy()
    plan.close()
    ref = oracle_mod.simulate(w.phantom.subset(idx), w.seq, output_mode="per_spin")
    assert_parity(rows, ref, "config 5b sampled dictionary rows")
    # every entry on its own scale as well: a dictionary row is used normalised
    for k in range(len(idx)):
        emax, _ = errors(rows[k], ref[k])
        assert emax <= TOL_MAX, f"entry {idx[k]}: max {emax:.3e}"


def test_full_config3_with_motion_experiment_d(B, oracle_mod):
    """Config 3m: the brain-like EPI with u_y = v_y t, v_y = 0.1 m/s, whole oracle."""
    import torch
    w = W.make("3m")
    plan = B.Plan(w.seq, **w.plan_kw)
    dev = B.phantom_to_device(w.phantom)
    vel = tuple(torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda() for a in w.velocity)
    Mxy = torch.zeros(w.phantom.n, 2, dtype=torch.float32, device="cuda")
    Mz = torch.zeros(w.phantom.n, dtype=torch.float32, device="cuda")
    sig = plan.simulate(*dev, Mxy=Mxy, Mz=Mz, velocity=vel)
    torch.cuda.synchronize()
    plan.close()
    ref, rxy, rz = oracle_mod.simulate(w.phantom, w.seq, velocity=w.velocity, dt_max=w.dt_max, return_state=True)
    m = Mxy.cpu().numpy()
    assert_parity(sig.cpu().numpy(), ref, "config 3m full-size signal")
    assert_parity(state_vec(m[:, 0] + 1j * m[:, 1], Mz.cpu().numpy()), state_vec(rxy, rz), "config 3m full-size final state")


def test_full_config4_with_8_coils_by_subset_and_superposition(B, oracle_mod):
    """Workload 4c (config 4 received by 8 coils) at full size: an evenly spaced subset against the
    oracle (every coil on its own scale), and superposition S_c(full) = S_c(subset) + S_c(complement) per coil, which
    ties the full-size launch (one pass of 8 coils, P = 2, 296 CTAs) to it."""
    import torch
    w = W.make("4c")
    n = w.phantom.n
    plan = B.Plan(w.seq, phase_mode=w.phase_mode, output_mode="sum")

    def run(idx):
        ph = w.phantom if idx is None else w.phantom.subset(idx)
        c = w.coils if idx is None else np.ascontiguousarray(w.coils[:, idx])
        sig = plan.simulate(*B.phantom_to_device(ph), coils=torch.from_numpy(c).cuda())
        torch.cuda.synchronize()
        return sig.cpu().numpy()

    full = run(None)
    assert full.shape == (8, 65536)
    assert np.array_equal(full.view(np.float32), run(None).view(np.float32)), "not bitwise reproducible"
    sub = np.linspace(0, n - 1, 192).astype(np.int64)
    s_sub = run(sub)
    ref = oracle_mod.simulate(w.phantom.subset(sub), w.seq, coils=w.coils[:, sub].astype(np.complex128))
    assert_parity(s_sub, ref, "config 4c subset, all coils")
    for c in range(8):
        assert_parity(s_sub[c], ref[c], f"config 4c subset, coil {c}")
    mask = np.ones(n, dtype=bool)
    mask[sub] = False
    s_rest = run(np.flatnonzero(mask))
    plan.close()
    for c in range(8):
        emax, nrmse = errors(s_sub[c].astype(np.complex128) + s_rest[c], full[c])
        assert emax < 5e-6 and nrmse < 1e-6, f"coil {c} superposition: max {emax:.3e} nrmse {nrmse:.3e}"
