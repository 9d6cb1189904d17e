"""Multi-coil receive on the GPU (bloch_simulate_coils; SURVEY.md 8(f) f2 "per-coil weights", reading C1) against the
oracle (pytest -m gpu).  Same acceptance as test_gpu_parity.py, per coil and normalised by the largest coil signal."""
import numpy as np
import pytest

from paper_2301_02702_b200 import workloads as W
from test_gpu_parity import B, assert_parity, errors  # noqa: F401  (B is a fixture)

pytestmark = pytest.mark.gpu


def coil_maps(ph, n_coils, seed=0):
    return W.coil_maps(ph, n_coils, seed=seed)


def run_coils(B, w, coils, want_state=False, **kw):
    import torch
    plan = B.Plan(w.seq, phase_mode=kw.pop("phase_mode", w.phase_mode), output_mode="sum", **kw)
    dev = B.phantom_to_device(w.phantom)
    n = w.phantom.n
    Mxy = torch.zeros(n, 2, dtype=torch.float32, device="cuda") if want_state else None
    Mz = torch.zeros(n, dtype=torch.float32, device="cuda") if want_state else None
    sig = plan.simulate(*dev, Mxy=Mxy, Mz=Mz, coils=torch.from_numpy(np.ascontiguousarray(coils)).cuda())
    torch.cuda.synchronize()
    out = sig.cpu().numpy()
    launches = B.bloch_plan_last_launches(plan.handle)
    plan.close()
    if want_state:
        m = Mxy.cpu().numpy()
        return out, m[:, 0] + 1j * m[:, 1], Mz.cpu().numpy(), launches
    return out


@pytest.mark.parametrize("name,n_coils,phase", [("1", 1, "fp32"), ("1", 4, "fp32"), ("2", 3, "fp32"), ("3", 8, "fp64"),
                                               ("4", 5, "fp32"), ("5", 2, "fp32")])
def test_small_configs_with_coils_match_oracle(B, oracle_mod, name, n_coils, phase):
    w = W.small(name)
    coils = coil_maps(w.phantom, n_coils, seed=n_coils)
    ref, rxy, rz = oracle_mod.simulate(w.phantom, w.seq, coils=coils.astype(np.complex128), return_state=True)
    got, gxy, gz, _ = run_coils(B, w, coils, want_state=True, phase_mode=phase)
    assert got.shape == ref.shape == (n_coils, w.seq.adc_t.size)
    assert_parity(got, ref, f"config {name}, {n_coils} coils")
    for c in range(n_coils):   # every coil on its own scale as well
        emax, nrmse = errors(got[c], ref[c])
        assert emax <= 1e-4 and nrmse <= 1e-5, f"coil {c}: max {emax:.3e} nrmse {nrmse:.3e}"
    assert_parity(np.concatenate([gxy, gz.astype(np.complex128)]), np.concatenate([rxy, rz.astype(np.complex128)]),
                  "final state with coils")


def test_uniform_coil_is_the_plain_signal_and_passes_are_independent(B):
    """One coil with weight 1 everywhere returns the plain signal; 9 coils (two passes of 8, the last with one coil)
    give the same rows as the same coils simulated in separate calls: bitwise when the pass width is the same
    (coils 0-7 alone), to rounding when it is not (4 coils per pass for up to 4 coils: other tile sizes)."""
    from test_gpu_parity import run_gpu
    w = W.small("4")
    ffma = {"coil_tc": 0}   # the per-block FFMA kernel (the tensor-core kernel / the whole-sequence kernel otherwise)
    n = w.phantom.n
    plain = run_gpu(B, w, path="per_block")
    one = run_coils(B, w, np.ones((1, n), dtype=np.complex64), options=ffma, path="per_block")
    emax, _ = errors(one[0], plain)
    assert emax < 2e-6, f"uniform coil vs plain: {emax:.3e}"
    coils = coil_maps(w.phantom, 9, seed=4)
    all9 = run_coils(B, w, coils, options=ffma, path="per_block")
    again = run_coils(B, w, coils, options=ffma, path="per_block")
    assert np.array_equal(all9.view(np.float32), again.view(np.float32)), "run-to-run not bitwise identical"
    first8 = run_coils(B, w, coils[:8], options=ffma, path="per_block")
    assert np.array_equal(all9[:8].view(np.float32), first8.view(np.float32))
    scale = np.abs(all9).max()
    first4 = run_coils(B, w, coils[:4], options=ffma, path="per_block")
    last1 = run_coils(B, w, coils[8:9], options=ffma, path="per_block")
    assert np.abs(all9[:4] - first4).max() / scale < 2e-6 and np.abs(all9[8:9] - last1).max() / scale < 2e-6


def test_coil_argument_errors_and_edge_cases(B):
    import torch
    w = W.small("1")
    n = w.phantom.n
    dev = B.phantom_to_device(w.phantom)
    coils = torch.ones(2, n, dtype=torch.complex64, device="cuda")
    for kw in (dict(output_mode="per_spin"),):
        plan = B.Plan(w.seq, **kw)
        ws = torch.empty(1 << 24, dtype=torch.uint8, device="cuda")
        sig = torch.empty(2, plan.info["n_adc"], dtype=torch.complex64, device="cuda")
        plan.upload()
        with pytest.raises(B.BlochError) as e:
            B.bloch_simulate_coils(plan.handle, n, *[t.data_ptr() for t in dev], 2, coils.data_ptr(), None, None, True,
                                   sig.data_ptr(), ws.data_ptr(), ws.numel())
        assert e.value.code == -1
        plan.close()
    plan = B.Plan(w.seq).upload()
    ws = torch.empty(1 << 24, dtype=torch.uint8, device="cuda")
    sig = torch.empty(2, plan.info["n_adc"], dtype=torch.complex64, device="cuda")
    with pytest.raises(B.BlochError):      # n_coils = 0
        B.bloch_simulate_coils(plan.handle, n, *[t.data_ptr() for t in dev], 0, coils.data_ptr(), None, None, True,
                               sig.data_ptr(), ws.data_ptr(), ws.numel())
    with pytest.raises(B.BlochError) as e:  # workspace sized without the coils
        small = B.bloch_plan_workspace_bytes(plan.handle, n)
        assert B.bloch_plan_workspace_bytes_coils(plan.handle, n, 2) > small
        B.bloch_simulate_coils(plan.handle, n, *[t.data_ptr() for t in dev], 2, coils.data_ptr(), None, None, True,
                               sig.data_ptr(), ws.data_ptr(), small)
    assert e.value.code == -4
    # zero spins: every coil's empty sum
    z = torch.zeros(0, dtype=torch.float32, device="cuda")
    out = plan.simulate(z, z, z, z, z, z, z, coils=torch.zeros(3, 0, dtype=torch.complex64, device="cuda"))
    torch.cuda.synchronize()
    assert out.shape == (3, plan.info["n_adc"]) and float(out.abs().max()) == 0.0
    plan.close()


def test_host_buffer_coil_entry_is_identical_to_the_device_entry(B):
    w = W.small("4")
    coils = coil_maps(w.phantom, 6, seed=2)
    dev_sig = run_coils(B, w, coils)
    plan = B.Plan(w.seq)
    ph = w.phantom
    mxy = np.zeros((ph.n, 2), dtype=np.float32); mz = np.zeros(ph.n, dtype=np.float32)
    h = plan.simulate_host(ph.x, ph.y, ph.z, ph.M0, ph.T1, ph.T2, ph.dw, Mxy=mxy, Mz=mz, coils=coils)
    plan.close()
    assert h.shape == (6, w.seq.adc_t.size)
    assert np.array_equal(h.view(np.float32), dev_sig.view(np.float32)), "host-buffer coil entry differs from device entry"
    assert np.abs(mz).max() > 0.1


@pytest.mark.parametrize("tc", [1, 2])
@pytest.mark.parametrize("name,n_coils", [("1", 5), ("4", 8), ("5", 11), ("2", 20), ("4", 37)])
def test_tensor_core_coil_kernel_matches_oracle(B, oracle_mod, name, n_coils, tc):
    """The tcgen05 / TMEM kernels (option coil_tc: 1 = csrc/coils_tc.cuh with 3xTF32 products, 2 = csrc/coils_h.cuh with FP16
    operand pieces, the default): contributions generated on the fly as the A operand in tensor memory, accumulators in
    TMEM.  Same acceptance as every other path; ragged sample tiles (n_adc not a multiple of 128), ragged 16-spin
    stages, 8, 16 and 32 coils per pass and two passes (37 coils) are all in these cases."""
    w = W.small(name)
    coils = coil_maps(w.phantom, n_coils, seed=10 + n_coils)
    ref, rxy, rz = oracle_mod.simulate(w.phantom, w.seq, coils=coils.astype(np.complex128), return_state=True)
    got, gxy, gz, launches = run_coils(B, w, coils, want_state=True, phase_mode="fp32", options={"coil_tc": tc}, path="per_block")
    emax, nrmse = assert_parity(got, ref, f"tensor-core coil kernel, config {name}, {n_coils} coils")
    print(f"coil_tc={tc} config {name} {n_coils} coils: max {emax:.3e} nrmse {nrmse:.3e}")
    for c in range(n_coils):
        emax, nrmse = errors(got[c], ref[c])
        assert emax <= 1e-4 and nrmse <= 1e-5, f"coil {c}: max {emax:.3e} nrmse {nrmse:.3e}"
    ffma = run_coils(B, w, coils, phase_mode="fp32", options={"coil_tc": 0}, path="per_block")
    emax, _ = errors(got, ffma)
    assert emax < 2e-5, f"tensor-core vs FFMA kernel: {emax:.3e}"   # TMEM accumulation is coarser than FFMA sums


@pytest.mark.parametrize("phase_mode,n_coils,wave", [("fp32", 3, False), ("fp64", 8, False), ("fp32", 6, True), ("fp64", 11, True)])
def test_coils_with_moving_spins(B, oracle_mod, phase_mode, n_coils, wave):
    """Coils x motion (PAPER.md:95 coil sensitivity, :96 motion field): S_c(t) = sum_i C_c(x_i) Mxy_i(t) with every spin
    moving, constant velocities or amplitudes on a shared waveform; the weights stay those of the spin's home position
    (they are per-spin inputs, reading C1).  Device and host entries; 11 coils = two passes of the 8-wide kernel."""
    import torch
    w = W.small("1")
    n = w.phantom.n
    rng = np.random.default_rng(50 + n_coils)
    coils = coil_maps(w.phantom, n_coils, seed=20 + n_coils)
    if wave:
        wt = np.arange(int(w.seq.t_end / 2.5e-4) + 2) * 2.5e-4
        wf = (wt, np.sin(2 * np.pi * 300.0 * wt))
        v = tuple(rng.uniform(-2e-3, 2e-3, n).astype(np.float32).astype(np.float64) for _ in range(3))
        kw = dict(motion="waveform", waveform=wf, dt_max=2e-5, max_speed_mps=4e-3)
    else:
        wf = None
        v = tuple(rng.uniform(-0.2, 0.2, n).astype(np.float32).astype(np.float64) for _ in range(3))
        kw = dict(motion="linear", dt_max=2e-5)
    ref, rxy, rz = oracle_mod.simulate(w.phantom, w.seq, coils=coils.astype(np.complex128), velocity=v, dt_max=2e-5,
                                       waveform=wf, return_state=True)
    plan = B.Plan(w.seq, phase_mode=phase_mode, **kw)
    dev = B.phantom_to_device(w.phantom)
    vel = tuple(torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda() for a in v)
    Mxy = torch.zeros(n, 2, dtype=torch.float32, device="cuda")
    Mz = torch.zeros(n, dtype=torch.float32, device="cuda")
    sig = plan.simulate(*dev, Mxy=Mxy, Mz=Mz, velocity=vel, coils=torch.from_numpy(coils).cuda())
    assert plan.status() == 0
    got = sig.cpu().numpy()
    assert_parity(got, ref, f"coils x motion {phase_mode} {n_coils} coils wave={wave}")
    for c in range(n_coils):
        emax, nrmse = errors(got[c], ref[c])
        assert emax <= 1e-4 and nrmse <= 1e-5, f"coil {c}: max {emax:.3e} nrmse {nrmse:.3e}"
    m = Mxy.cpu().numpy()
    assert_parity(np.concatenate([m[:, 0] + 1j * m[:, 1], Mz.cpu().numpy().astype(np.complex128)]),
                  np.concatenate([rxy, rz.astype(np.complex128)]), "final state, coils x motion")
    ph = w.phantom
    host = plan.simulate_host(ph.x, ph.y, ph.z, ph.M0, ph.T1, ph.T2, ph.dw, velocity=v, coils=coils)
    assert np.array_equal(host.view(np.float32), got.view(np.float32)), "host entry differs from the device entry"
    static = oracle_mod.simulate(w.phantom, w.seq, coils=coils.astype(np.complex128))
    assert errors(ref, static)[0] > 1e-2, "the motion must change the signal for the test to mean anything"
    plan.close()


def run_coils_path(B, w, coils, path, want_state=True, **kw):
    """Signal, final state and what the plan reports about the launch, on a given path."""
    import torch
    plan = B.Plan(w.seq, path=path, phase_mode="fp32", output_mode="sum", **kw)
    dev = B.phantom_to_device(w.phantom)
    n = w.phantom.n
    Mxy = torch.zeros(n, 2, dtype=torch.float32, device="cuda") if want_state else None
    Mz = torch.zeros(n, dtype=torch.float32, device="cuda") if want_state else None
    sig = plan.simulate(*dev, Mxy=Mxy, Mz=Mz, coils=torch.from_numpy(np.ascontiguousarray(coils)).cuda())
    torch.cuda.synchronize()
    out = dict(sig=sig.cpu().numpy(), launches=B.bloch_plan_last_launches(plan.handle),
               fused=B.bloch_plan_last_kernel(plan.handle, "fused")["name"])
    if want_state:
        m = Mxy.cpu().numpy()
        out.update(mxy=m[:, 0] + 1j * m[:, 1], mz=Mz.cpu().numpy())
    plan.close()
    return out


@pytest.mark.parametrize("name,n_coils", [("2", 1), ("2", 4), ("2", 7), ("5", 3), ("5", 8), ("1", 5), ("4", 6)])
def test_coils_inside_the_whole_sequence_kernel(B, oracle_mod, name, n_coils):
    """f2 x (a5-a8 in one launch): up to 8 receive coils are summed per coil inside seq_kernel<0, NC> (ring of partial
    rows per coil, sum over the CTAs in the launch).  Against the oracle per coil, and against the per-block kernels."""
    w = W.small(name)
    coils = coil_maps(w.phantom, n_coils, seed=10 + n_coils)
    ref, rxy, rz = oracle_mod.simulate(w.phantom, w.seq, coils=coils.astype(np.complex128), return_state=True)
    f = run_coils_path(B, w, coils, "fused")
    nc = 4 if n_coils <= 4 else 8
    assert f["fused"] == f"seq_kernel<0, {nc}>", f["fused"]
    assert f["launches"] == 4, f["launches"]          # pack, pack_coils, seq_kernel, unpack
    assert f["sig"].shape == ref.shape == (n_coils, w.seq.adc_t.size)
    emax, nrmse = assert_parity(f["sig"], ref, f"config {name}, {n_coils} coils, whole-sequence kernel")
    print(f"config {name} fused with {n_coils} coils: max {emax:.3e} nrmse {nrmse:.3e}")
    for c in range(n_coils):
        e, r = errors(f["sig"][c], ref[c])
        assert e <= 1e-4 and r <= 1e-5, f"coil {c}: max {e:.3e} nrmse {r:.3e}"
    assert_parity(np.concatenate([f["mxy"], f["mz"].astype(np.complex128)]),
                  np.concatenate([rxy, rz.astype(np.complex128)]), "final state")
    p = run_coils_path(B, w, coils, "per_block")
    assert p["fused"] == ""
    assert np.array_equal(f["mxy"], p["mxy"]) and np.array_equal(f["mz"], p["mz"]), "final state differs bitwise between paths"
    e, _ = errors(f["sig"], p["sig"])
    assert e < 2e-5, f"fused vs per-block coil signals: {e:.3e}"
    for _ in range(4):   # integer tickets, fixed summation order: bitwise reproducible
        g = run_coils_path(B, w, coils, "fused", want_state=False)
        assert np.array_equal(g["sig"].view(np.float32), f["sig"].view(np.float32))


def test_fused_coils_limits_and_auto_choice(B):
    w = W.small("5")
    # more than 8 coils: AUTO runs the per-block kernels, a forced FUSED plan is refused
    c9 = coil_maps(w.phantom, 9, seed=3)
    a = run_coils_path(B, w, c9, "auto", want_state=False)
    assert a["fused"] == "" and a["sig"].shape[0] == 9
    with pytest.raises(B.BlochError) as e:
        run_coils_path(B, w, c9, "fused", want_state=False)
    assert e.value.code == -1
    # up to 8: AUTO takes the whole-sequence kernel where it would without coils (unless 8 coils meet blocks large
    # enough for the tcgen05 kernel: 2^24 (spin, sample) pairs), and both agree
    c8 = c9[:8]
    a8 = run_coils_path(B, w, c8, "auto", want_state=False)
    assert a8["fused"] == "seq_kernel<0, 8>"
    e, _ = errors(a8["sig"], a["sig"][:8])
    assert e < 2e-5
    # a uniform coil is the plain signal of the same path (same summation order per sample: close, not bitwise --
    # the plain kernel shares one ex2 between adjacent samples)
    import torch
    one = np.ones((1, w.phantom.n), dtype=np.complex64)
    u = run_coils_path(B, w, one, "fused", want_state=False)
    plan = B.Plan(w.seq, path="fused", phase_mode="fp32")
    plain = plan.simulate(*B.phantom_to_device(w.phantom))
    torch.cuda.synchronize()
    e, _ = errors(u["sig"][0], plain.cpu().numpy())
    plan.close()
    assert e < 2e-6, f"{e:.3e}"


@pytest.mark.parametrize("m_scale,w_scale,init", [(1.0, 1.0, "big"), (2.0 ** -14, 2.0 ** 17, "eq"), (3.0e4, 7.0e-6, "eq"),
                                                 (1.0, 0.0, "eq")])
def test_fp16_tensor_core_coil_kernel_scales_its_operands(B, oracle_mod, m_scale, w_scale, init):
    """The FP16 tensor-core coil kernel (csrc/coils_h.cuh) scales both MMA operands by powers of two taken from measured
    maxima (FP16 has 5 exponent bits): magnetisations and coil weights far from 1, an initial state larger than M0, and
    all-zero weights must come out as the oracle has them, on the scale of the result."""
    import dataclasses
    w = W.small("4")
    ph = dataclasses.replace(w.phantom, M0=(w.phantom.M0 * m_scale).astype(np.float32).astype(np.float64))
    w = dataclasses.replace(w, phantom=ph)
    coils = (coil_maps(ph, 8, seed=5) * w_scale).astype(np.complex64)
    state = None
    if init == "big":   # |M(0)| = 3 M0, tipped: the bound on |M| is max(M0, |M(0)|)
        state = ((2.0 * ph.M0 * np.exp(0.3j * np.arange(ph.n))).astype(np.complex64), (2.2 * ph.M0).astype(np.float32))
    ref = oracle_mod.simulate(ph, w.seq, coils=coils.astype(np.complex128),
                              state=None if state is None else (state[0].astype(np.complex128), state[1].astype(np.float64)))
    import torch
    plan = B.Plan(w.seq, path="per_block", phase_mode="fp32", options={"coil_tc": 2})
    dev = B.phantom_to_device(ph)
    kw = {}
    if state is not None:
        kw = dict(Mxy=torch.view_as_real(torch.from_numpy(state[0]).cuda()).contiguous(), Mz=torch.from_numpy(state[1]).cuda(),
                  init_equilibrium=False)
    got = plan.simulate(*dev, coils=torch.from_numpy(coils).cuda(), **kw).cpu().numpy()
    assert B.bloch_plan_last_kernel(plan.handle, "signal")["name"] == "signal_coils_h_kernel<8>"
    plan.close()
    if w_scale == 0.0:
        assert not got.any() and not np.asarray(ref).any()
        return
    emax, nrmse = assert_parity(got, ref, f"fp16 coil kernel, M0 x {m_scale:g}, weights x {w_scale:g}, init {init}")
    print(f"fp16 coil kernel, M0 x {m_scale:g}, weights x {w_scale:g}, init {init}: max {emax:.3e} nrmse {nrmse:.3e}")
