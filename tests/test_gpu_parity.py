"""GPU-vs-oracle parity through the C-ABI (run on the B200 box: pytest -m gpu).

Acceptance (BASELINE.json north_star; NRMSE as reading G17, normalised by the oracle signal's maximum as the
paper normalises its own errors):
    max|S_gpu - S_ref| / max|S_ref| <= 1e-4      and      sqrt(mean|S_gpu - S_ref|^2) / max|S_ref| <= 1e-5
"""
import numpy as np
import pytest

from paper_2301_02702_b200 import workloads as W
from seqtools import phantom, seq

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


def assert_parity(got, ref, what=""):
    emax, nrmse = errors(got, ref)
    assert emax <= TOL_MAX and nrmse <= TOL_NRMSE, f"{what}: max {emax:.3e} nrmse {nrmse:.3e}"
    return emax, nrmse


def run_gpu(B, w, *, state=None, want_state=False, **plan_kw):
    import torch
    kw = dict(phase_mode=w.phase_mode, output_mode=w.output_mode)
    kw.update(plan_kw)
    plan = B.Plan(w.seq, **kw)
    dev = B.phantom_to_device(w.phantom)
    n = w.phantom.n
    Mxy = Mz = None
    init = True
    if state is not None:
        Mxy = torch.view_as_real(torch.from_numpy(np.asarray(state[0], dtype=np.complex64)).cuda()).contiguous()
        Mz = torch.from_numpy(np.asarray(state[1], dtype=np.float32)).cuda()
        init = False
    elif want_state:
        Mxy = torch.zeros(n, 2, dtype=torch.float32, device="cuda")
        Mz = torch.zeros(n, dtype=torch.float32, device="cuda")
    sig = plan.simulate(*dev, Mxy=Mxy, Mz=Mz, init_equilibrium=init)
    torch.cuda.synchronize()
    out = sig.cpu().numpy()
    plan.close()
    if want_state:
        m = Mxy.cpu().numpy()
        return out, m[:, 0] + 1j * m[:, 1], Mz.cpu().numpy()
    return out


@pytest.mark.parametrize("name", ["1", "2", "3", "4", "5", "5b"])
def test_small_configs_match_oracle(B, oracle_mod, name):
    w = W.small(name)
    ref, rxy, rz = oracle_mod.simulate(w.phantom, w.seq, output_mode=w.output_mode, return_state=True)
    got, gxy, gz = run_gpu(B, w, want_state=True)
    assert got.shape == ref.shape
    assert_parity(got, ref, f"config {name} signal")
    # final magnetisation, same two measures on the (Mxy, Mz) arrays
    assert_parity(np.concatenate([gxy, gz.astype(np.complex128)]), np.concatenate([rxy, rz.astype(np.complex128)]),
                  f"config {name} final state")


@pytest.mark.parametrize("name", ["1", "4"])
def test_phase_variants_agree_with_oracle(B, oracle_mod, name):
    w = W.small(name)
    ref = oracle_mod.simulate(w.phantom, w.seq)
    for mode in ("fp32", "fp64"):
        assert_parity(run_gpu(B, w, phase_mode=mode), ref, f"config {name} phase {mode}")


def test_block_cut_and_launch_shapes_do_not_change_the_answer(B, oracle_mod):
    """max_block_points cuts precession blocks (PAPER.md:171 Nblocks); the result must not depend on it
    beyond rounding (exactness of the precession regime, :132)."""
    w = W.small("4")
    ref = oracle_mod.simulate(w.phantom, w.seq)
    for mbp in (0, 257, 64):
        assert_parity(run_gpu(B, w, max_block_points=mbp), ref, f"max_block_points={mbp}")


def test_bitwise_reproducible_and_host_path_identical(B):
    import torch
    w = W.small("4")
    a = run_gpu(B, w)
    b = run_gpu(B, w)
    assert np.array_equal(a.view(np.float32), b.view(np.float32)), "run-to-run not bitwise identical"
    plan = B.Plan(w.seq)
    ph = w.phantom
    h = plan.simulate_host(ph.x, ph.y, ph.z, ph.M0, ph.T1, ph.T2, ph.dw)
    plan.close()
    assert np.array_equal(a.view(np.float32), h.view(np.float32)), "host-buffer entry differs from device entry"


def test_initial_state_roundtrip_resume(B, oracle_mod):
    """Final magnetisation out + initial magnetisation in = resume: two half sequences chained through the
    state equal one full run (checkpoint/resume row)."""
    rng = np.random.default_rng(7)
    n = 301
    ph = phantom(x=rng.uniform(-.1, .1, n), y=rng.uniform(-.1, .1, n), z=rng.uniform(-.01, .01, n),
                 M0=rng.uniform(.5, 1, n), T1=rng.uniform(.3, 2, n), T2=rng.uniform(.03, .3, n),
                 dw=rng.uniform(-300, 300, n))
    ph = W._phantom(ph.x, ph.y, ph.z, ph.M0, ph.T1, ph.T2, ph.dw)
    rf = (np.arange(100) * 1e-5, np.full(100, 1e-5), np.full(100, 4e-6), np.full(100, 1e-6))
    g = {0: ([1.2e-3, 1.4e-3, 3e-3, 3.2e-3], [0, 8e-3, 8e-3, 0])}
    adc = 1.5e-3 + np.arange(100) * 1e-5
    s = seq(g=g, rf=rf, adc=adc, t_end=4e-3, dt_rf_max=1e-5)
    state0 = (rng.normal(0, .3, n) + 1j * rng.normal(0, .3, n), rng.uniform(-1, 1, n))
    state0 = (state0[0].astype(np.complex64).astype(np.complex128), state0[1].astype(np.float32).astype(np.float64))
    w = W.Workload("resume", ph, s)
    ref, rxy, rz = oracle_mod.simulate(ph, s, state=state0, return_state=True)
    got, gxy, gz = run_gpu(B, w, state=state0, want_state=True)
    assert_parity(got, ref, "signal from a supplied initial state")
    assert_parity(np.concatenate([gxy, gz.astype(np.complex128)]), np.concatenate([rxy, rz.astype(np.complex128)]),
                  "final state from a supplied initial state")


def test_edge_cases(B, oracle_mod):
    import torch
    # (1) no ADC at all: only the final magnetisation
    ph = phantom(x=[0.01, -0.02, 0.03], T1=[1.0, 0.5, 2.0], T2=[0.1, 0.05, 0.2], dw=[10.0, -20.0, 0.0])
    s = seq(rf=([1e-4], [2e-4], [3e-5], [0.0]), t_end=2e-3, dt_rf_max=1e-5)
    w = W.Workload("noadc", ph, s)
    _, rxy, rz = oracle_mod.simulate(ph, s, return_state=True)
    got, gxy, gz = run_gpu(B, w, want_state=True)
    assert got.shape == (0,)
    assert_parity(np.concatenate([gxy, gz.astype(np.complex128)]), np.concatenate([rxy, rz.astype(np.complex128)]), "no-ADC")
    # (2) no RF at all, ADC at t = 0 and at t_end, a supplied transverse state
    s = seq(g={1: ([0, 1e-3, 2e-3], [0, 5e-3, 0])}, adc=[0.0, 5e-4, 2e-3], t_end=2e-3)
    st = (np.array([0.5 + 0.25j, -0.125j, 1.0]), np.array([0.0, 0.5, -1.0]))
    ph = phantom(y=[0.01, -0.02, 0.03], T1=[1.0, 0.5, 2.0], T2=[0.1, 0.05, 0.2], dw=[10.0, -20.0, 0.0])
    ref = oracle_mod.simulate(ph, s, state=st)
    got = run_gpu(B, W.Workload("norf", ph, s), state=st)
    assert_parity(got, ref, "no-RF, ADC on both ends")
    # (3) one spin, one-step hard 90 (|w| = pi/2 > polynomial range -> sqrt/sincos branch), per-spin output
    b1 = (np.pi / 2) / (W.GAMMA * 1e-4)
    s = seq(rf=([0.0], [1e-4], [b1], [0.0]), adc=[1e-4, 3e-4], t_end=1e-3, dt_rf_max=1.0)
    ph = phantom(T1=[1.0], T2=[0.1])
    ref = oracle_mod.simulate(ph, s, output_mode="per_spin")
    got = run_gpu(B, W.Workload("one", ph, s, output_mode="per_spin"))
    assert got.shape == (1, 2)
    assert_parity(got, ref, "single spin, one-step hard pulse")
    # (4) zero spins: the empty sum
    plan = B.Plan(s).upload()
    z = torch.zeros(0, dtype=torch.float32, device="cuda")
    out = plan.simulate(z, z, z, z, z, z, z)
    torch.cuda.synchronize()
    assert out.shape == (2,) and float(out.abs().max()) == 0.0
    plan.close()


def test_superposition_over_spin_shards(B):
    """S(A u B) = S(A) + S(B) (invariant I3): the multi-GPU sharding rule of DESIGN.md, checked on one GPU."""
    w = W.small("4")
    n = w.phantom.n
    full = run_gpu(B, w)
    a = run_gpu(B, W.Workload("a", w.phantom.subset(slice(0, n // 2)), w.seq))
    b = run_gpu(B, W.Workload("b", w.phantom.subset(slice(n // 2, n)), w.seq))
    emax, nrmse = errors(a + b, full)
    assert emax < 2e-6 and nrmse < 5e-7
