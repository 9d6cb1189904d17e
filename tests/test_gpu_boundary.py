"""Boundary behaviour of the C-ABI on the device (VERDICT r1 "close the boundary holes"):
what bloch_simulate finds out about the phantom it is given -- invalid relaxation times, non-finite values, a phantom
larger than the extents the plan was told to assume -- is reported loudly, never silently computed through."""
import math

import numpy as np
import pytest

from paper_2301_02702_b200 import workloads as W
from seqtools import seq

pytestmark = pytest.mark.gpu

EINVAL, ERANGE = -1, -10


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


def readout_sequence():
    """Hard 90 + 1.5 ms of 10 mT/m: k reaches 681 turns/m (170 turns at 0.25 m, 409 turns at 0.6 m)."""
    g = {0: ([2e-4, 3e-4, 1.8e-3, 1.9e-3], [0, 10e-3, 10e-3, 0]), 1: ([2e-4, 3e-4, 1.8e-3, 1.9e-3], [0, -3e-3, -3e-3, 0])}
    rf = ([0.0], [1e-4], [(math.pi / 2) / (W.GAMMA * 1e-4)], [0.0])
    return seq(g=g, rf=rf, adc=3e-4 + (np.arange(300) + 0.5) * 5e-6, t_end=2e-3, dt_rf_max=1e-5)


def body_phantom(n, half, seed):
    rng = np.random.default_rng(seed)
    return W._phantom(rng.uniform(-half, half, n), rng.uniform(-half, half, n), rng.uniform(-0.01, 0.01, n),
                      rng.uniform(0.5, 1, n), rng.uniform(0.3, 2, n), rng.uniform(0.03, 0.3, n),
                      2 * np.pi * rng.uniform(-200, 200, n))


@pytest.mark.parametrize("field,value", [("T2", 0.0), ("T2", -0.05), ("T1", float("nan")), ("T1", float("inf")),
                                         ("T2", float("nan")), ("x", float("nan")), ("dw", float("inf"))])
def test_invalid_phantom_values_fail_loudly(B, field, value):
    import torch
    w = W.small("1")
    ph = w.phantom
    arrs = {k: np.array(getattr(ph, k), dtype=np.float32) for k in ("x", "y", "z", "M0", "T1", "T2", "dw")}
    arrs[field][517] = value
    order = ("x", "y", "z", "M0", "T1", "T2", "dw")
    plan = B.Plan(w.seq)
    good = B.phantom_to_device(ph)
    bad = tuple(torch.from_numpy(arrs[k]).cuda() for k in order)
    # (1) explicit collection
    plan.simulate(*bad)
    with pytest.raises(B.BlochError) as e:
        plan.status()
    assert e.value.code == EINVAL and ("T1 or T2" in str(e.value)) == (field in ("T1", "T2"))
    assert plan.status() == 0                      # reported once, then cleared
    # (2) nobody collects: the NEXT call on the plan fails instead of running, once
    plan.simulate(*bad)
    torch.cuda.synchronize()
    with pytest.raises(B.BlochError) as e:
        plan.simulate(*good)
    assert e.value.code == EINVAL
    sig = plan.simulate(*good)
    assert plan.status() == 0 and np.isfinite(sig.cpu().numpy().view(np.float32)).all()
    # (3) the host-buffer entry checks before it returns
    with pytest.raises(B.BlochError) as e:
        plan.simulate_host(*[arrs[k] for k in order])
    assert e.value.code == EINVAL
    plan.simulate_host(*[np.asarray(getattr(ph, k), dtype=np.float32) for k in order])
    plan.close()


def test_large_body_phantom_under_auto_needs_declared_extents_and_then_matches_the_oracle(B, oracle_mod):
    """A 0.8 x 0.8 m phantom (|x| up to 0.57 m) on a sequence whose k reaches 681 turns/m: the default extents
    (0.25 m) let AUTO choose fp32 phase, and the simulation reports BLOCH_ERANGE instead of silently losing phase
    precision; with max_extent_m declared AUTO takes fp64 phase accumulation and the result matches the oracle."""
    import torch
    s = readout_sequence()
    ph = body_phantom(3000, 0.4, 5)
    dev = B.phantom_to_device(ph)
    ref = oracle_mod.simulate(ph, s)

    plan = B.Plan(s)                                   # AUTO, default extents -> fp32 phase
    assert plan.info["phase_mode"] == B.PHASE_FP32
    plan.simulate(*dev)
    with pytest.raises(B.BlochError) as e:
        plan.status()
    assert e.value.code == ERANGE and "max |x|" in str(e.value)
    small = body_phantom(3000, 0.15, 6)                # inside the declared extents: fine on the same plan
    got_small = plan.simulate(*B.phantom_to_device(small)).cpu().numpy()
    assert plan.status() == 0
    emax, nrmse = errors(got_small, oracle_mod.simulate(small, s))
    assert emax <= 1e-4 and nrmse <= 1e-5
    with pytest.raises(B.BlochError) as e:             # the host entry reports it as its return code
        plan.simulate_host(ph.x, ph.y, ph.z, ph.M0, ph.T1, ph.T2, ph.dw)
    assert e.value.code == ERANGE
    plan.close()

    plan = B.Plan(s, max_extent_m=0.6)                 # declared: AUTO resolves to fp64 phase
    assert plan.info["phase_mode"] == B.PHASE_FP64
    got = plan.simulate(*dev).cpu().numpy()
    assert plan.status() == 0
    plan.close()
    emax, nrmse = errors(got, ref)
    print(f"0.8 m phantom, AUTO with max_extent_m = 0.6: max {emax:.3e} nrmse {nrmse:.3e}")
    assert emax <= 1e-4 and nrmse <= 1e-5

    plan = B.Plan(s, phase_mode="fp32")                # forced fp32: the caller took the precision on, no check
    plan.simulate(*dev)
    assert plan.status() == 0
    plan.close()


def test_off_resonance_and_speed_extents_are_measured_too(B):
    import torch
    s = readout_sequence()
    ph = body_phantom(2000, 0.1, 7)
    plan = B.Plan(s, motion="linear", dt_max=1e-4)
    dev = B.phantom_to_device(ph)
    fat = list(dev)
    fat[6] = dev[6] * 0 + 2 * math.pi * 200e3           # 200 kHz "metal": 2e5 Hz x 1.9 ms = 380 turns
    plan.simulate(*fat)
    with pytest.raises(B.BlochError) as e:
        plan.status()
    assert e.value.code == ERANGE
    v = tuple(torch.full((ph.n,), val, dtype=torch.float32, device="cuda") for val in (400.0, 0.0, 0.0))
    plan.simulate(*dev, velocity=v)                     # 400 m/s x first moment (~0.7 turn s/m) on top of 172 turns
    with pytest.raises(B.BlochError) as e:
        plan.status()
    assert e.value.code == ERANGE
    slow = tuple(torch.full((ph.n,), val, dtype=torch.float32, device="cuda") for val in (0.1, 0.0, 0.0))
    plan.simulate(*dev, velocity=slow)
    assert plan.status() == 0
    plan.close()


def test_wrong_output_buffers_are_rejected_by_the_binding(B):
    import torch
    w = W.small("1")
    plan = B.Plan(w.seq)
    dev = B.phantom_to_device(w.phantom)
    n, n_adc = w.phantom.n, plan.info["n_adc"]
    with pytest.raises(AssertionError):
        plan.simulate(*dev, signal=torch.empty(n_adc - 1, dtype=torch.complex64, device="cuda"))
    with pytest.raises(AssertionError):
        plan.simulate(*dev, signal=torch.empty(n_adc, dtype=torch.complex128, device="cuda"))
    with pytest.raises(AssertionError):
        plan.simulate(*dev, Mxy=torch.zeros(n, 2, dtype=torch.float64, device="cuda"),
                      Mz=torch.zeros(n, dtype=torch.float32, device="cuda"))
    with pytest.raises(AssertionError):
        plan.simulate(*dev, Mxy=torch.zeros(2 * n, 2, dtype=torch.float32, device="cuda")[::2],
                      Mz=torch.zeros(n, dtype=torch.float32, device="cuda"))
    ph = w.phantom
    host = [np.asarray(getattr(ph, k), dtype=np.float32) for k in ("x", "y", "z", "M0", "T1", "T2", "dw")]
    with pytest.raises(AssertionError):
        plan.simulate_host(*host, signal=np.empty(n_adc, dtype=np.complex128))
    with pytest.raises(AssertionError):
        plan.simulate_host(*host, Mxy=np.zeros((n, 2), dtype=np.float64), Mz=np.zeros(n, dtype=np.float32))
    plan.close()
