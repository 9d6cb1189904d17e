"""GROUPED output (isochromat ensembles per voxel / dictionary entry)
on the GPU against the oracle's definition.  Same acceptance as the other parity tests."""
import numpy as np
import pytest

from paper_2301_02702_b200 import workloads as W

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


def gpu(B, w, ph=None, **kw):
    import torch
    ph = w.phantom if ph is None else ph
    k = dict(w.plan_kw)
    k.update(kw)
    plan = B.Plan(w.seq, **k)
    sig = plan.simulate(*B.phantom_to_device(ph))
    torch.cuda.synchronize()
    out = sig.cpu().numpy()
    plan.close()
    return out


def test_ensemble_dictionary_small(B, oracle_mod):
    w = W.small("5c")
    got = gpu(B, w)
    ref = oracle_mod.simulate(w.phantom, w.seq, output_mode="grouped", group_size=w.group_size)
    assert got.shape == ref.shape == (41, 40)
    emax, nrmse = errors(got, ref)
    print(f"5c small: max {emax:.3e} nrmse {nrmse:.3e}")
    assert emax <= TOL_MAX and nrmse <= TOL_NRMSE
    for g in range(got.shape[0]):              # every entry on its own scale
        assert errors(got[g], ref[g])[0] <= TOL_MAX, g


@pytest.mark.parametrize("gs", [1, 7, 32, 100, 1001])
def test_group_sizes_against_per_spin_and_sum(B, oracle_mod, gs):
    """Group sizes below, at and above a warp; gs = 1 is PER_SPIN, gs = n_spins is SUM_ALL; readouts of many
    samples per block exercise the per-point loop."""
    w = W.small("4")
    n = (w.phantom.n // gs) * gs
    ph = w.phantom.subset(slice(0, n))
    got = gpu(B, w, ph, output_mode="grouped", group_size=gs)
    ref = oracle_mod.simulate(ph, w.seq, output_mode="grouped", group_size=gs)
    assert got.shape == (n // gs, ref.shape[1])
    emax, nrmse = errors(got, ref)
    print(f"gs={gs}: max {emax:.3e} nrmse {nrmse:.3e}")
    assert emax <= TOL_MAX and nrmse <= TOL_NRMSE
    again = gpu(B, w, ph, output_mode="grouped", group_size=gs)
    assert np.array_equal(got.view(np.float32), again.view(np.float32)), "not bitwise reproducible"


def test_grouped_argument_errors(B):
    import torch
    w = W.small("5c")
    with pytest.raises(B.BlochError):
        B.Plan(w.seq, output_mode="grouped", group_size=0)
    plan = B.Plan(w.seq, output_mode="grouped", group_size=5).upload()
    dev = B.phantom_to_device(w.phantom.subset(slice(0, 7)))
    with pytest.raises(B.BlochError) as e:
        plan.simulate(*dev)
    assert e.value.code == -1
    plan.close()


def test_full_ensemble_dictionary_sampled_entries(B, oracle_mod):
    """Config 5c at full size (10,000 entries x 64 isochromats, 1000 TRs): sampled entries against the oracle."""
    import torch
    w = W.make("5c")
    plan = B.Plan(w.seq, **w.plan_kw)
    sig = plan.simulate(*B.phantom_to_device(w.phantom))
    torch.cuda.synchronize()
    plan.close()
    gs = w.group_size
    assert tuple(sig.shape) == (w.phantom.n // gs, 1000)
    rng = np.random.default_rng(13)
    ent = np.sort(rng.choice(w.phantom.n // gs, 6, replace=False))
    idx = (ent[:, None] * gs + np.arange(gs)[None, :]).ravel()
    ref = oracle_mod.simulate(w.phantom.subset(idx), w.seq, output_mode="grouped", group_size=gs)
    got = sig[torch.from_numpy(ent).cuda()].cpu().numpy()
    emax, nrmse = errors(got, ref)
    print(f"5c full sampled entries: max {emax:.3e} nrmse {nrmse:.3e}")
    assert emax <= TOL_MAX and nrmse <= TOL_NRMSE
