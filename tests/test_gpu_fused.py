"""The whole-sequence kernel (BLOCH_PATH_FUSED, csrc/seq.cuh) against the oracle and against the per-block path
(pytest -m gpu).  Same acceptance as test_gpu_parity.py; in addition the final magnetisation must be BITWISE
equal to the per-block path (both round the state to one float per component at the same places) and the
signal may differ from it only by the order of the fixed-order sums."""
import numpy as np
import pytest

from paper_2301_02702_b200 import workloads as W
from seqtools import phantom, seq
from test_gpu_parity import B, assert_parity, errors, run_gpu  # noqa: F401  (B is a fixture)

pytestmark = pytest.mark.gpu


def both_paths(B, w, **kw):
    out = {}
    for path in ("per_block", "fused"):
        out[path] = run_gpu(B, w, want_state=True, path=path, phase_mode="fp32", **kw)
    return out


@pytest.mark.parametrize("name", ["1", "2", "4", "5"])
def test_small_configs_fused_matches_oracle_and_per_block(B, oracle_mod, name):
    w = W.small(name)
    ref, rxy, rz = oracle_mod.simulate(w.phantom, w.seq, return_state=True)
    out = both_paths(B, w)
    sig, mxy, mz = out["fused"]
    assert_parity(sig, ref, f"config {name} fused signal")
    assert_parity(np.concatenate([mxy, mz.astype(np.complex128)]), np.concatenate([rxy, rz.astype(np.complex128)]),
                  f"config {name} fused state")
    assert np.array_equal(mxy, out["per_block"][1]) and np.array_equal(mz, out["per_block"][2]), \
        "final magnetisation differs bitwise between the paths"
    emax, _ = errors(sig, out["per_block"][0])
    assert emax < 2e-6, f"fused vs per-block signal: {emax:.3e}"


def test_auto_picks_fused_only_where_it_qualifies(B):
    w = W.small("5")
    n = w.phantom.n

    def uses(n_spins=n, **kw):
        plan = B.Plan(w.seq, **kw)
        u = B.bloch_plan_uses_fused(plan.handle, n_spins)
        plan.close()
        return u

    assert uses(phase_mode="fp32")                                  # excitation-heavy, few spins: fused
    assert not uses(phase_mode="fp32", path="per_block")
    assert not uses(phase_mode="fp64")                              # fp64 phase: per-block only
    assert not uses(phase_mode="fp32", output_mode="per_spin")
    assert not uses(n_spins=1_000_000, phase_mode="fp32")          # more than 29 warps of spins per SM
    assert not uses(n_spins=1_000_000, phase_mode="fp32", path="fused")
    # 120,000 spins = 26 RF warps per SM leave room for 4 signal warps only: allowed when forced, not what AUTO picks
    assert not uses(n_spins=120_000, phase_mode="fp32")
    assert uses(n_spins=120_000, phase_mode="fp32", path="fused")
    # readout-heavy sequence (config 1: 50 RF steps, 1024 ADC samples): AUTO stays per-block, FUSED can be forced
    w1 = W.small("1")
    p = B.Plan(w1.seq, phase_mode="fp32")
    assert not B.bloch_plan_uses_fused(p.handle, w1.phantom.n)
    p.close()
    p = B.Plan(w1.seq, phase_mode="fp32", path="fused")
    assert B.bloch_plan_uses_fused(p.handle, w1.phantom.n)
    p.close()


def test_forced_fused_on_an_unqualified_plan_is_an_error(B):
    import torch
    w = W.small("5")
    plan = B.Plan(w.seq, phase_mode="fp64", path="fused")
    dev = B.phantom_to_device(w.phantom)
    with pytest.raises(B.BlochError) as e:
        plan.simulate(*dev)
    torch.cuda.synchronize()
    assert e.value.code == -1   # BLOCH_EINVAL
    with pytest.raises(B.BlochError):
        B.bloch_plan_set_path(plan.handle, 7)
    plan.close()


@pytest.mark.parametrize("n", [1, 31, 33, 148 * 32 + 1, 9000])
def test_ragged_spin_counts(B, oracle_mod, n):
    """Chunks of 32 / 64 spins per CTA, a last CTA with one spin, fewer CTAs than SMs."""
    w = W.small("5")
    rng = np.random.default_rng(n)
    ph = W._phantom(rng.uniform(-.1, .1, n), rng.uniform(-.1, .1, n), np.zeros(n), rng.uniform(.5, 1, n),
                    rng.uniform(.3, 2, n), rng.uniform(.03, .3, n), rng.uniform(-100, 100, n))
    ww = W.Workload("ragged", ph, w.seq)
    ref, rxy, rz = oracle_mod.simulate(ph, w.seq, return_state=True)
    out = both_paths(B, ww)
    assert_parity(out["fused"][0], ref, f"n={n} signal")
    assert np.array_equal(out["fused"][1], out["per_block"][1]) and np.array_equal(out["fused"][2], out["per_block"][2])
    assert_parity(np.concatenate([out["fused"][1], out["fused"][2].astype(np.complex128)]),
                  np.concatenate([rxy, rz.astype(np.complex128)]), f"n={n} state")


def test_fused_is_bitwise_reproducible_and_independent_of_the_signal_warp_count(B):
    w = W.small("2")
    a = run_gpu(B, w, path="fused", phase_mode="fp32")
    b = run_gpu(B, w, path="fused", phase_mode="fp32")
    assert np.array_equal(a.view(np.float32), b.view(np.float32)), "run-to-run not bitwise identical"
    # the partial of a CTA is one thread's sum over the chunk's spins in index order whatever the number of signal
    # warps (only which thread owns which sample changes; the P = 1/2/4 choice moves with it, hence a tolerance)
    for base, extra in ((1, 0), (0, 1), (3, 2), (5, 0)):
        c = run_gpu(B, w, path="fused", phase_mode="fp32", options={"seq_sig_base": base, "seq_sig_extra": extra})
        emax, _ = errors(c, a)
        assert emax < 2e-6, f"signal warps base {base} extra {extra}: {emax:.3e}"


def test_fused_supplied_state_precession_first_and_no_adc(B, oracle_mod):
    rng = np.random.default_rng(11)
    n = 777
    ph = W._phantom(rng.uniform(-.1, .1, n), rng.uniform(-.1, .1, n), rng.uniform(-.005, .005, n),
                    rng.uniform(.5, 1, n), rng.uniform(.3, 2, n), rng.uniform(.03, .3, n), rng.uniform(-300, 300, n))
    st = (rng.normal(0, .3, n) + 1j * rng.normal(0, .3, n), rng.uniform(-1, 1, n))
    st = (st[0].astype(np.complex64).astype(np.complex128), st[1].astype(np.float32).astype(np.float64))
    # (1) a readout BEFORE the first pulse (the supplied transverse state is what it sees), two pulses, a block
    # without ADC between them, ADC samples after the last pulse up to t_end
    rf_t = np.concatenate([1e-3 + np.arange(200) * 1e-6, 3e-3 + np.arange(300) * 1e-6])
    rf = (rf_t, np.full(500, 1e-6), np.full(500, 5e-6), np.linspace(-2e-6, 2e-6, 500))
    g = {0: ([0, 1e-4, 9e-4, 1e-3], [0, 6e-3, 6e-3, 0]), 2: ([2.9e-3, 3e-3, 3.3e-3, 3.4e-3], [0, 5e-3, 5e-3, 0]),
         1: ([3.5e-3, 3.6e-3, 5e-3], [0, 4e-3, 4e-3])}
    adc = np.concatenate([1e-4 + np.arange(70) * 1e-5, 3.6e-3 + np.arange(139) * 1e-5, [5e-3]])
    s = seq(g=g, rf=rf, adc=adc, t_end=5e-3)
    ref, rxy, rz = oracle_mod.simulate(ph, s, state=st, return_state=True)
    got, gxy, gz = run_gpu(B, W.Workload("pre", ph, s), state=st, want_state=True, path="fused", phase_mode="fp32")
    assert_parity(got, ref, "precession first, supplied state: signal")
    assert_parity(np.concatenate([gxy, gz.astype(np.complex128)]), np.concatenate([rxy, rz.astype(np.complex128)]),
                  "precession first, supplied state: final state")
    # (2) no ADC at all
    s = seq(g=g, rf=rf, t_end=5e-3)
    _, rxy, rz = oracle_mod.simulate(ph, s, return_state=True)
    got, gxy, gz = run_gpu(B, W.Workload("noadc", ph, s), want_state=True, path="fused", phase_mode="fp32")
    assert got.shape == (0,)
    assert_parity(np.concatenate([gxy, gz.astype(np.complex128)]), np.concatenate([rxy, rz.astype(np.complex128)]),
                  "no ADC: final state")
    # (3) no RF at all (the producer warp has nothing to stream)
    s = seq(g=g, adc=adc, t_end=5e-3)
    ref = oracle_mod.simulate(ph, s, state=st)
    got = run_gpu(B, W.Workload("norf", ph, s), state=st, path="fused", phase_mode="fp32")
    assert_parity(got, ref, "no RF: signal")


def test_fused_mixed_tiles_and_tiers(B, oracle_mod):
    """General (gradient-ramp) and compact step tiles, a change of step length, and spins far enough off-centre
    for tier 1 next to tier-0 warps in the same CTA."""
    dts = np.concatenate([np.full(300, 1e-6), np.full(40, 5e-6), np.full(150, 1e-6)])
    t0 = 1e-4 + np.concatenate([[0.0], np.cumsum(dts)[:-1]])
    rng = np.random.default_rng(5)
    b1, b1i = rng.uniform(-4e-6, 4e-6, dts.size), rng.uniform(-4e-6, 4e-6, dts.size)
    t_rf_end = t0[-1] + dts[-1]
    g = {0: ([0.0, 3e-4, 5e-4, 9e-4], [0, 12e-3, -6e-3, 0]), 2: ([0.0, 2e-4, 6e-4, 1.2e-3], [10e-3, 10e-3, -9e-3, 0])}
    adc = t_rf_end + 1e-5 + np.arange(333) * 3e-6
    s = seq(g=g, rf=(t0, dts, b1, b1i), adc=adc, t_end=2.5e-3, dt_rf_max=1.0)
    n = 2500
    z = np.concatenate([rng.uniform(-.002, .002, n // 2), rng.uniform(-.08, .08, n - n // 2)])
    ph = W._phantom(rng.uniform(-.1, .1, n), rng.uniform(-.1, .1, n), z, rng.uniform(.5, 1, n),
                    rng.uniform(.3, 2, n), rng.uniform(.03, .3, n), rng.uniform(-300, 300, n))
    ref, rxy, rz = oracle_mod.simulate(ph, s, return_state=True)
    out = both_paths(B, W.Workload("mixed", ph, s))
    assert_parity(out["fused"][0], ref, "mixed tiles: signal")
    assert np.array_equal(out["fused"][1], out["per_block"][1]) and np.array_equal(out["fused"][2], out["per_block"][2])
    assert_parity(np.concatenate([out["fused"][1], out["fused"][2].astype(np.complex128)]),
                  np.concatenate([rxy, rz.astype(np.complex128)]), "mixed tiles: state")


def test_fused_per_spin_dictionary_mode(B, oracle_mod):
    """PER_SPIN plans with a few samples per block (an MRF dictionary: one sample per TR) run as ONE launch: the
    thread that owns the spin evaluates its samples itself.  Against the oracle and the per-block path."""
    w = W.small("5b")
    ref, rxy, rz = oracle_mod.simulate(w.phantom, w.seq, output_mode="per_spin", return_state=True)
    out = {}
    for path in ("per_block", "fused"):
        out[path] = run_gpu(B, w, want_state=True, path=path, phase_mode="fp32")
    sig, mxy, mz = out["fused"]
    assert sig.shape == ref.shape == (w.phantom.n, w.seq.adc_t.size)
    assert_parity(sig, ref, "dictionary, whole-sequence kernel")
    assert_parity(np.concatenate([mxy, mz.astype(np.complex128)]), np.concatenate([rxy, rz.astype(np.complex128)]),
                  "dictionary final state")
    assert np.array_equal(mxy, out["per_block"][1]) and np.array_equal(mz, out["per_block"][2])
    emax, _ = errors(sig, out["per_block"][0])
    assert emax < 2e-6
    plan = B.Plan(w.seq, phase_mode="fp32", output_mode="per_spin")
    assert B.bloch_plan_uses_fused(plan.handle, w.phantom.n)          # AUTO takes it
    assert B.bloch_plan_uses_fused(plan.handle, 100_000)              # 22 RF warps per SM
    assert not B.bloch_plan_uses_fused(plan.handle, 640_000)
    plan.close()
    w5 = W.small("5")                                                 # 300 samples per block: not this way
    plan = B.Plan(w5.seq, phase_mode="fp32", output_mode="per_spin", path="fused")
    assert not B.bloch_plan_uses_fused(plan.handle, w5.phantom.n)
    plan.close()


def test_fused_is_race_free_over_many_runs(B):
    """The roles of the whole-sequence kernel meet only at mbarriers; a missing edge would show up as run-to-run
    differences.  25 runs each with 1, 2 and 3 signal warps per sub-partition (plus the balancing extras) (different interleavings of the roles), all bitwise equal
    per configuration, signal and final state."""
    w = W.small("5")
    for nw in (1, 2, 3):
        first = None
        for _ in range(25):
            sig, mxy, mz = run_gpu(B, w, want_state=True, path="fused", phase_mode="fp32", options={"seq_sig_base": nw})
            cur = (sig.view(np.float32).copy(), mxy.view(np.float32).copy(), mz.copy())
            if first is None:
                first = cur
            else:
                assert all(np.array_equal(a, b) for a, b in zip(first, cur)), f"{nw} signal warps: runs differ"
