"""Full-size parity of configs 4, 5 and 5b against the WHOLE fp64 oracle (north_star: "all five configs match the
fp64 oracle"; "full-size parity is still computed once per config and cached by input hash").

The expected values are `tests/golden/fullsize_config{4,5,5b}.npz`, written by `tests/golden/make_fullsize_golden.py`,
which imports only `oracle` and the seeded input generators: every spin, every interval of the step-by-step
integrator (1.6e11 / 2.0e11 / 2.0e11 spin*steps).  Here the full-size GPU run -- in the launch configuration bench.py
times -- is compared with them ELEMENT BY ELEMENT (Fig 3: signal per ADC sample summed over all spins;
:244: errors normalised by the reference maximum), after checking that the goldens belong to exactly these inputs.
Configs 1-3 and 3m run the whole oracle live (tests/test_gpu_fullsize.py).
"""
import importlib.util
import os

import numpy as np
import pytest

from paper_2301_02702_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_MAX = 1e-4      # BASELINE.json north_star
TOL_NRMSE = 1e-5    # reading G17

_spec = importlib.util.spec_from_file_location(
    "make_fullsize_golden", os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "make_fullsize_golden.py"))
G = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(G)


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


def load_golden(name, w):
    path = G.golden_path(name)
    assert os.path.exists(path), f"{path} missing: run tests/golden/make_fullsize_golden.py {name}"
    z = np.load(path)
    assert str(z["input_sha256"]) == G.input_sha256(w), "golden was written for other inputs (seed / generator changed)"
    assert int(z["n_spins"]) == w.phantom.n
    return z


def run_full(B, w, **plan_kw):
    import torch
    plan = B.Plan(w.seq, **dict(w.plan_kw, **plan_kw))
    n = w.phantom.n
    Mxy = torch.zeros(n, 2, dtype=torch.float32, device="cuda")
    Mz = torch.zeros(n, dtype=torch.float32, device="cuda")
    sig = plan.simulate(*B.phantom_to_device(w.phantom), Mxy=Mxy, Mz=Mz)
    assert plan.status() == 0
    info, fused = plan.info, B.bloch_plan_uses_fused(plan.handle, n)
    plan.close()
    m = Mxy.cpu().numpy()
    return sig, m[:, 0] + 1j * m[:, 1], Mz.cpu().numpy(), info, fused


def state_vec(mxy, mz):
    return np.concatenate([np.asarray(mxy, dtype=np.complex128), np.asarray(mz, dtype=np.complex128)])


@pytest.mark.parametrize("name", ["4", "5"])
def test_full_size_signal_and_state_against_the_whole_oracle(B, name):
    """Config 4: 1,000,000 spins x 163,285 intervals, 65,536 ADC samples (per-block path).  Config 5: 65,536 spins x
    3,060,777 intervals, 1,024,000 ADC samples (whole-sequence kernel).  Every ADC sample against the oracle's sum
    over ALL spins; the final magnetisation of every (config 4: every 8th) spin."""
    w = W.make(name)
    z = load_golden(name, w)
    sig, mxy, mz, info, fused = run_full(B, w)
    assert info["n_intervals"] == int(z["n_intervals"])
    assert fused == (name == "5")
    got = sig.cpu().numpy()
    assert got.shape == z["signal"].shape
    assert_parity(got, z["signal"], f"config {name} full-size signal vs whole oracle ({w.phantom.n} spins)")
    st = int(z["state_stride"])
    assert_parity(state_vec(mxy[::st], mz[::st]), state_vec(z["Mxy"], z["Mz"]),
                  f"config {name} final magnetisation vs whole oracle ({len(z['Mz'])} spins)")


def test_full_size_signal_on_the_other_path(B):
    """Config 5 on the per-block path (2001 RF / signal launches) against the same whole-oracle golden."""
    w = W.make("5")
    z = load_golden("5", w)
    sig, mxy, mz, _, fused = run_full(B, w, path="per_block")
    assert not fused
    assert_parity(sig.cpu().numpy(), z["signal"], "config 5 per-block path vs whole oracle")
    assert_parity(state_vec(mxy, mz), state_vec(z["Mxy"], z["Mz"]), "config 5 per-block final magnetisation")


def test_full_size_dictionary_every_row_against_the_whole_oracle(B):
    """Config 5b: all 100,000 dictionary entries x every 25th TR (40 of the 1000 columns; a TR's sample depends on
    the whole history before it), and the final magnetisation of every entry after 1e6 RF steps; every entry also
    on its own scale, since a dictionary row is used normalised."""
    import torch
    w = W.make("5b")
    z = load_golden("5b", w)
    sig, mxy, mz, info, fused = run_full(B, w)
    assert tuple(sig.shape) == (w.phantom.n, info["n_adc"]) and fused
    cols = z["columns"]
    assert np.array_equal(cols, G.columns_5b(info["n_adc"]))
    got = sig[:, torch.from_numpy(cols).cuda()].cpu().numpy()
    ref = z["signal"]
    assert got.shape == ref.shape
    assert_parity(got, ref, "config 5b, 100,000 rows x 40 TRs vs whole oracle")
    row_err = np.abs(got.astype(np.complex128) - ref).max(axis=1) / np.abs(ref).max(axis=1)
    print(f"config 5b worst row on its own scale: {row_err.max():.3e} (entry {int(row_err.argmax())})")
    assert row_err.max() <= TOL_MAX
    assert_parity(state_vec(mxy, mz), state_vec(z["Mxy"], z["Mz"]), "config 5b final magnetisation, every entry")


def test_full_size_config5_with_8_coils_inside_the_whole_sequence_kernel(B, oracle_mod):
    """Workload 5x8 (config 5 received by 8 coils, f2 x whole-sequence kernel) at full size: 65,536 spins, 1,024,000
    samples x 8 coils in ONE launch.  (1) The coil maps are normalised to add up to one at every spin, so the sum of
    the 8 coil signals is the plain signal (reading C1 is linear in the weights) -- compared with the WHOLE oracle of
    config 5, every sample.  (2) A 96-spin subset against the oracle with coils, every coil on its own scale.
    (3) Superposition per coil S_c(full) = S_c(subset) + S_c(complement), which ties the full-size launch to (2)."""
    import torch
    w = W.make("5x8")
    z = load_golden("5", W.make("5"))       # same phantom and sequence: the oracle of config 5, all 65,536 spins
    n = w.phantom.n
    # complex maps that add up to 1 + 0i at every spin: magnitudes normalised, imaginary parts made zero-sum over coils
    m = np.abs(w.coils).astype(np.float64)
    m /= m.sum(axis=0, keepdims=True)
    q = m * np.sin(np.angle(w.coils))
    q -= q.mean(axis=0, keepdims=True)
    coils = (m + 1j * q).astype(np.complex64)
    # forced: with 8 coils and 6.7e7 (spin, sample) pairs per block AUTO prefers the per-block tcgen05 kernel
    plan = B.Plan(w.seq, phase_mode="fp32", path="fused")

    def run(idx):
        ph = w.phantom if idx is None else w.phantom.subset(idx)
        c = coils if idx is None else np.ascontiguousarray(coils[:, idx])
        sig = plan.simulate(*B.phantom_to_device(ph), coils=torch.from_numpy(c).cuda())
        torch.cuda.synchronize()
        return sig.cpu().numpy(), B.bloch_plan_last_kernel(plan.handle, "fused")["name"], \
            B.bloch_plan_last_launches(plan.handle)

    full, kernel, launches = run(None)
    assert kernel == "seq_kernel<0, 8>" and launches == 3, (kernel, launches)
    assert full.shape == (8, 1_024_000)
    assert np.array_equal(full.view(np.float32), run(None)[0].view(np.float32)), "not bitwise reproducible"
    total = full.astype(np.complex128).sum(axis=0)
    resid = np.abs(coils.astype(np.complex128).sum(axis=0) - 1.0).max()   # complex64 rounding of the normalised maps
    assert resid < 1e-6
    assert_parity(total, z["signal"], "config 5x8: sum of the 8 coil signals vs whole oracle of config 5 (65536 spins)")
    sub = np.linspace(0, n - 1, 96).astype(np.int64)
    s_sub = run(sub)[0]
    ref = oracle_mod.simulate(w.phantom.subset(sub), w.seq, coils=coils[:, sub].astype(np.complex128))
    assert_parity(s_sub, ref, "config 5x8 subset, all coils")
    for c in range(8):
        assert_parity(s_sub[c], ref[c], f"config 5x8 subset, coil {c}")
    mask = np.ones(n, dtype=bool)
    mask[sub] = False
    s_rest = run(np.flatnonzero(mask))[0]
    plan.close()
    for c in range(8):
        emax, nrmse = errors(s_sub[c].astype(np.complex128) + s_rest[c], full[c])
        assert emax < 5e-6 and nrmse < 1e-6, f"coil {c} superposition: max {emax:.3e} nrmse {nrmse:.3e}"
