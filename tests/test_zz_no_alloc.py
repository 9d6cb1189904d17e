"""bloch_simulate_static (include/bloch.h): the simulation on the library's OWN static device workspace, for callers
that cannot allocate device memory.  Checked against the existing path (bloch_simulate with a caller workspace) on
calls made one after the other on the shared array, plus the size limit and the refusals.  pytest -m gpu; collected
last on purpose (file name), self-contained so that it also passes alone in a fresh process."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_MAX = 1e-4      # BASELINE.json north_star, as tests/test_gpu_parity.py
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
    scale = max(np.abs(ref).max(), 1e-30)
    d = np.abs(got - ref)
    return d.max() / scale, np.sqrt(np.mean(d ** 2)) / scale


class Case:
    """One workload with its plan, device phantom and output tensors for both entry points."""

    def __init__(self, B, name, **plan_kw):
        import torch
        from paper_2301_02702_b200 import workloads as W
        self.w = W.small(name)
        kw = dict(phase_mode=self.w.phase_mode, output_mode=self.w.output_mode)
        kw.update(plan_kw)
        self.plan = B.Plan(self.w.seq, **kw).upload()
        self.dev = B.phantom_to_device(self.w.phantom)
        self.n = self.w.phantom.n
        self.shape = self.plan._signal_shape(self.n)
        self.torch = torch

    def outputs(self):
        t = self.torch
        return (t.full(self.shape, 7.0, dtype=t.complex64, device="cuda"),  # sentinel: every element must be written
                t.zeros(self.n, 2, dtype=t.float32, device="cuda"), t.zeros(self.n, dtype=t.float32, device="cuda"))

    def existing(self):
        sig, mxy, mz = self.outputs()
        self.plan.simulate(*self.dev, Mxy=mxy, Mz=mz, signal=sig)
        self.torch.cuda.synchronize()
        return sig.cpu().numpy(), mxy.cpu().numpy(), mz.cpu().numpy()

    def static_enqueue(self):
        sig, mxy, mz = self.outputs()
        self.plan.simulate_static(*self.dev, signal=sig, Mxy=mxy, Mz=mz)
        return sig, mxy, mz


def check(case, got, ref, what):
    g = [t.cpu().numpy() for t in got]
    for a, b, part in zip(g, ref, ("signal", "Mxy", "Mz")):
        emax, nrmse = errors(a, b)
        assert emax <= TOL_MAX and nrmse <= TOL_NRMSE, f"{what} {part}: max {emax:.3e} nrmse {nrmse:.3e}"
        # same kernels, same launch shapes, same workspace layout: the static entry point is bitwise the existing one
        assert np.array_equal(a, b), f"{what} {part}: not bitwise equal to bloch_simulate"
    print(f"{what}: {case.n} spins, static workspace result bitwise equal to bloch_simulate")


def test_static_workspace_matches_existing_path_on_calls_in_a_row(B):
    import torch
    # per-block two-pass sum (4), whole-sequence kernel with tickets (2), fp64 phase (3), per-spin rows (5b)
    cases = [Case(B, "4", phase_mode="fp32"), Case(B, "2", phase_mode="fp32"), Case(B, "3"), Case(B, "5b")]
    refs = [c.existing() for c in cases]
    # every pair (a, b): call a then b on the shared array with no synchronisation in between (one stream serialises
    # them); b finds a's partial rows, tickets and spin records in the array and must not be affected by them
    for i, a in enumerate(cases):
        for j, b in enumerate(cases):
            ga = a.static_enqueue()
            gb = b.static_enqueue()
            torch.cuda.synchronize()
            check(a, ga, refs[i], f"first call (config {a.w.name})")
            check(b, gb, refs[j], f"second call in a row (config {b.w.name} after {a.w.name})")
    # the same call twice in a row, then once more after the array has held another plan's data
    c = cases[1]
    g1, g2 = c.static_enqueue(), c.static_enqueue()
    torch.cuda.synchronize()
    check(c, g1, refs[1], "repeat 1")
    check(c, g2, refs[1], "repeat 2")
    for c in cases:
        c.plan.close()


def test_static_entry_point_allocates_no_device_memory(B):
    import torch
    c = Case(B, "2", phase_mode="fp32")
    out = c.outputs()
    for _ in range(2):  # warm-up: module load, kernel attributes
        c.plan.simulate_static(*c.dev, signal=out[0], Mxy=out[1], Mz=out[2])
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    stats0 = torch.cuda.memory_allocated()
    for _ in range(5):
        c.plan.simulate_static(*c.dev, signal=out[0], Mxy=out[1], Mz=out[2])
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, f"device memory shrank by {free0 - free1} B across 5 calls"
    assert torch.cuda.memory_allocated() == stats0
    c.plan.close()


def test_static_entry_point_rejects_what_it_cannot_serve(B):
    import torch
    from paper_2301_02702_b200 import workloads as W
    c = Case(B, "4", phase_mode="fp32")
    # beyond the limit: 2,000,000 spins x 48 B of packed records alone pass 32 MiB
    n_big = 2_000_000
    need = B.bloch_plan_workspace_bytes_coils(c.plan.handle, n_big, 0)
    assert need > B.STATIC_WORKSPACE_BYTES
    arrs = [torch.ones(n_big, dtype=torch.float32, device="cuda") for _ in range(7)]
    sig = torch.full(c.shape, 7.0, dtype=torch.complex64, device="cuda")
    with pytest.raises(B.BlochError) as e:
        c.plan.simulate_static(*arrs, signal=sig)
    assert e.value.code == -4 and "static" in str(e.value) and str(B.STATIC_WORKSPACE_BYTES) in str(e.value), str(e.value)
    torch.cuda.synchronize()
    assert bool((sig == 7.0).all()), "a refused call must enqueue nothing"
    # the largest size that fits does run (and the one after it is refused): the limit is exact
    lo, hi = c.n, n_big
    while hi - lo > 1:
        mid = (lo + hi) // 2
        if B.bloch_plan_workspace_bytes_coils(c.plan.handle, mid, 0) <= B.STATIC_WORKSPACE_BYTES:
            lo = mid
        else:
            hi = mid
    c.plan.simulate_static(*[a[:lo] for a in arrs], signal=sig)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(torch.view_as_real(sig)).all()) and not bool((sig == 7.0).any())
    with pytest.raises(B.BlochError):
        c.plan.simulate_static(*[a[:hi] for a in arrs], signal=sig)
    print(f"limit: {lo} spins of this plan fit {B.STATIC_WORKSPACE_BYTES} B, {hi} do not")
    # profiling taps create CUDA events: refused; switched off again: served
    out = c.outputs()
    B.bloch_plan_set_profiling(c.plan.handle, True)
    with pytest.raises(B.BlochError) as e:
        c.plan.simulate_static(*c.dev, signal=out[0])
    assert e.value.code == -1
    B.bloch_plan_set_profiling(c.plan.handle, False)
    c.plan.simulate_static(*c.dev, signal=out[0])
    # motion plans: refused
    wm = W.small("3m")
    pm = B.Plan(wm.seq, **wm.plan_kw).upload()
    dm = B.phantom_to_device(wm.phantom)
    sm = torch.zeros(pm._signal_shape(wm.phantom.n), dtype=torch.complex64, device="cuda")
    with pytest.raises(B.BlochError) as e:
        pm.simulate_static(*dm, signal=sm)
    assert e.value.code == -1
    # no spins: the sum over nothing, no workspace touched
    z = [torch.empty(0, dtype=torch.float32, device="cuda") for _ in range(7)]
    c.plan.simulate_static(*z, signal=out[0])
    torch.cuda.synchronize()
    assert bool((out[0] == 0).all())
    pm.close()
    c.plan.close()
