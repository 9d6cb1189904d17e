"""Host logic of the C-ABI library (no GPU): symbols, planner counts, error paths."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

from paper_2301_02702_b200 import build as bl
from paper_2301_02702_b200 import workloads as W
from seqtools import seq

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    bl.build()
    from paper_2301_02702_b200 import bloch
    return bloch


def test_library_exports_every_declared_symbol(B):
    hdr = open(os.path.join(ROOT, "include", "bloch.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(bloch_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(B.EXPORTS)
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_2301_02702_b200", "libbloch_b200.so"))
    for name in declared:
        assert hasattr(lib, name), name
    assert B.bloch_version() >= 100
    assert B.bloch_strerror(-3)


@pytest.mark.parametrize("name", ["1", "2", "3", "4", "5", "5b"])
def test_plan_counts_match_oracle_grid(B, oracle_mod, name):
    w = W.small(name)
    h = B.bloch_plan_create(w.seq, phase_mode=w.phase_mode, output_mode=w.output_mode)
    try:
        info = B.bloch_plan_get_info(h)
        t, G, rf, adc = oracle_mod.grid(w.seq)
        assert info["n_intervals"] == len(t) - 1
        assert info["n_rf_steps"] == int(rf.sum())
        assert info["n_adc"] == len(w.seq.adc_t)
        assert info["n_eval_points"] == info["n_adc"] + (info["n_blocks"] - info["n_rf_blocks"])
        assert info["table_bytes"] % 256 == 0
        assert B.bloch_plan_workspace_bytes(h, w.phantom.n) >= 48 * w.phantom.n
        assert info["phase_mode"] == (B.PHASE_FP64 if w.phase_mode == "fp64" else B.PHASE_FP32)
    finally:
        B.bloch_plan_destroy(h)


def test_plan_error_paths(B):
    ok = dict(g={0: ([1e-3, 2e-3], [0.0, 0.0])}, rf=([0.0], [1e-4], [1e-6], [0.0]), adc=[5e-4], t_end=3e-3)
    h = B.bloch_plan_create(seq(**ok))
    B.bloch_plan_destroy(h)
    bad = dict(ok); bad["g"] = {0: ([2e-3, 1e-3], [0.0, 0.0])}
    with pytest.raises(B.BlochError) as e:
        B.bloch_plan_create(seq(**bad))
    assert e.value.code == -2
    bad = dict(ok); bad["rf"] = ([0.0, 5e-5], [1e-4, 1e-4], [1e-6, 1e-6], [0.0, 0.0])   # overlap
    with pytest.raises(B.BlochError) as e:
        B.bloch_plan_create(seq(**bad))
    assert e.value.code == -2
    bad = dict(ok); bad["t_end"] = -1.0
    with pytest.raises(B.BlochError) as e:
        B.bloch_plan_create(seq(**bad))
    assert e.value.code == -1
    bad = dict(ok); bad["adc"] = [4e-3]                 # beyond t_end
    with pytest.raises(B.BlochError) as e:
        B.bloch_plan_create(seq(**bad))
    assert e.value.code == -1
    with pytest.raises(B.BlochError) as e:              # simulate before upload
        h = B.bloch_plan_create(seq(**ok))
        try:
            B.bloch_simulate(h, 4, 1, 1, 1, 1, 1, 1, 1, None, None, True, 1, 256, 1 << 20)
        finally:
            B.bloch_plan_destroy(h)
    assert e.value.code == -7


def test_adc_on_rf_boundary_is_served_by_precession_block(B):
    s = seq(rf=([1e-3], [1e-4], [1e-6], [0.0]), adc=[1e-3, 1.1e-3, 2e-3], t_end=3e-3, dt_rf_max=1e-5)
    h = B.bloch_plan_create(s)
    info = B.bloch_plan_get_info(h)
    B.bloch_plan_destroy(h)
    assert info["n_blocks"] == 3 and info["n_rf_blocks"] == 1 and info["n_rf_steps"] == 10
    assert info["n_adc"] == 3 and info["max_block_adc"] == 2


def test_max_block_points_splits_precession_blocks(B):
    adc = np.linspace(1e-3, 9e-3, 100)
    s = seq(adc=adc, t_end=10e-3)
    h = B.bloch_plan_create(s, max_block_points=16)
    info = B.bloch_plan_get_info(h)
    B.bloch_plan_destroy(h)
    assert info["n_blocks"] == 7 and info["max_block_adc"] == 16


def test_rf_increment_form_equals_eq9():
    """The RF kernel applies Eq 9 as M+ = M + a (w x M) + b (w x (w x M)) (kernels.cuh).  Check that
    identity against Eq 6-9 written out with complex spinors, in fp64 numpy."""
    rng = np.random.default_rng(0)
    for _ in range(200):
        w = rng.normal(0, 1.0, 3) * rng.choice([1e-4, 1e-2, 1.0])
        M = rng.normal(0, 1, 3)
        t = np.linalg.norm(w)
        phi = -t                                       # Eq 8 with w = gamma B dt
        nxy, nz = (w[0] + 1j * w[1]) / t, w[2] / t
        al = math.cos(phi / 2) - 1j * nz * math.sin(phi / 2)
        be = -1j * nxy * math.sin(phi / 2)
        mxy = M[0] + 1j * M[1]
        mxy2 = 2 * np.conj(al) * be * M[2] + np.conj(al) ** 2 * mxy - be ** 2 * np.conj(mxy)
        mz2 = (abs(al) ** 2 - abs(be) ** 2) * M[2] - 2 * (al * be * np.conj(mxy)).real
        a, b = -math.sin(t) / t, (1 - math.cos(t)) / t ** 2
        u = np.cross(w, M)
        got = M + a * u + b * np.cross(w, u)
        np.testing.assert_allclose(got, [mxy2.real, mxy2.imag, mz2], rtol=0, atol=1e-14)


@pytest.mark.parametrize("name,dt_max", [("1", 2e-5), ("2", 1e-4), ("4", 5e-6)])
def test_motion_plan_refines_like_the_oracle(B, oracle_mod, name, dt_max):
    """With motion every interval is limited to dt_max; the planner's grid must be the oracle's."""
    w = W.small(name)
    h0 = B.bloch_plan_create(w.seq)
    h1 = B.bloch_plan_create(w.seq, motion="linear", dt_max=dt_max)
    try:
        i0, i1 = B.bloch_plan_get_info(h0), B.bloch_plan_get_info(h1)
        t, _, rf, _ = oracle_mod.grid(w.seq, dt_max=dt_max)
        assert i1["n_intervals"] == len(t) - 1 and i1["n_rf_steps"] == int(rf.sum())
        assert i1["n_intervals"] > i0["n_intervals"] and i1["motion_mode"] == 1 and i0["motion_mode"] == 0
        assert i1["table_bytes"] > i0["table_bytes"]      # first-moment records
        assert i1["n_adc"] == i0["n_adc"] and i1["n_blocks"] == i0["n_blocks"]
    finally:
        B.bloch_plan_destroy(h0)
        B.bloch_plan_destroy(h1)
    with pytest.raises(B.BlochError):
        B.bloch_plan_create(w.seq, motion=7)


def test_scanner_limits_are_checked_when_given(B):
    """the scanner carries B0, G_max, S_max; they bound the waveforms, not the arithmetic."""
    # trapezoid: 30 mT/m reached in 200 us (150 T/m/s), then a 10 us edge of 3000 T/m/s
    s = seq(g={1: ([1e-3, 1.2e-3, 2e-3, 2.01e-3], [0.0, 30e-3, 30e-3, 0.0])}, adc=[1.5e-3], t_end=3e-3)
    for kw in ({}, dict(G_max=60e-3, S_max=5000.0), dict(G_max=30e-3), dict(S_max=3000.0)):
        h = B.bloch_plan_create(s, **kw)       # within limits (equality allowed) or limits not given
        B.bloch_plan_destroy(h)
    for kw in (dict(G_max=29e-3), dict(S_max=200.0), dict(G_max=60e-3, S_max=2999.0)):
        with pytest.raises(B.BlochError) as e:
            B.bloch_plan_create(s, **kw)
        assert e.value.code == -9, kw
    # the generators' own sequences respect the limits they were built for (60 mT/m, 200 T/m/s ramps)
    from paper_2301_02702_b200 import workloads as W
    for name in ("1", "2", "3"):
        h = B.bloch_plan_create(W.small(name).seq, G_max=60e-3)
        B.bloch_plan_destroy(h)


def test_planner_flags_all_cartesian_blocks_for_the_recurrence_kernel(B):
    """Block::lin_pts is visible through n_launches: a flagged block whose length is not a multiple of 16 costs one more
    launch (its tail).  Flagged: equally spaced samples on a plateau (also with motion, where mu' is a parabola).
    Not flagged: samples running through the ramp (k' quadratic), unequal spacing, fewer than 20 groups."""
    def launches(adc, g, **kw):
        s = seq(g=g, adc=adc, t_end=3.1e-2)
        h = B.bloch_plan_create(s, **kw)
        info = B.bloch_plan_get_info(h)
        B.bloch_plan_destroy(h)
        return info["n_launches"]

    plateau = {0: ([1e-4, 2e-4, 3e-2], [0, 5e-3, 5e-3])}
    t0, dw = 2.5e-4, 5e-6
    base = launches(t0 + np.arange(2048) * dw, plateau)
    assert launches(t0 + np.arange(2053) * dw, plateau) == base + 1                      # tail of 5 samples
    assert launches(t0 + np.arange(2053) * dw, plateau, motion="linear", dt_max=1e-5) == \
        launches(t0 + np.arange(2048) * dw, plateau, motion="linear", dt_max=1e-5) + 1
    assert launches(1.5e-4 + np.arange(2053) * dw, plateau) == base                      # first samples on the ramp
    jit = t0 + np.arange(2053) * dw
    jit[1000] += 1e-9
    assert launches(jit, plateau) == base                                                # one sample 1 ns late
    assert launches(t0 + np.arange(317) * dw, plateau) == base                           # 19 groups: too short
    assert launches(t0 + np.arange(325) * dw, plateau) == base + 1                       # 20 groups + tail of 5


def test_plan_options_are_plan_state_not_environment(B):
    """Kernel selection is set per plan (bloch_plan_set_option), echoed by bloch_plan_get_info, validated, and the
    library's sources read no environment variable."""
    h = B.bloch_plan_create(W.small("1").seq)
    try:
        info = B.bloch_plan_get_info(h)
        assert info["options"] == {"signal_lin": 1, "signal_p": 0, "signal_fixed_cta": 0, "signal_ctas_per_sm": 4,
                                   "rf_threads": 0, "rf_spins": 0, "coil_tc": -1, "seq_sig_extra": -1,
                                   "seq_sig_base": -1, "seq_items_x4": 0, "rf_const": 1}
        B.bloch_plan_set_option(h, "signal_lin", 0)
        B.bloch_plan_set_option(h, B.OPTIONS.index("signal_p"), 4)
        assert B.bloch_plan_get_option(h, "signal_lin") == 0 and B.bloch_plan_get_option(h, "signal_p") == 4
        info = B.bloch_plan_get_info(h)
        assert info["options"]["signal_lin"] == 0 and info["options"]["signal_p"] == 4
        for key, bad in (("signal_p", 3), ("signal_ctas_per_sm", 0), ("rf_threads", 48), ("coil_tc", 3), (99, 0),
                         ("rf_spins", 3)):
            with pytest.raises(B.BlochError) as e:
                B.bloch_plan_set_option(h, key, bad)
            assert e.value.code == -1
        B.bloch_plan_set_path(h, "per_block")
        assert B.bloch_plan_get_info(h)["path"] == B.PATHS["per_block"]
    finally:
        B.bloch_plan_destroy(h)
    csrc = os.path.join(ROOT, "paper_2301_02702_b200", "csrc")
    for fn in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, fn)).read(), f"{fn} reads the environment"


def test_phase_mode_auto_follows_the_declared_extents(B):
    """BLOCH_PHASE_AUTO bounds the block-relative phase with the extents the caller declares in bloch_sim_params
    (defaults 0.25 m / 1 kHz / 1 m/s): k = 42.58e6 x 10 mT/m x 1.6 ms (ramps included) = 681 turns/m is 170 turns at
    0.25 m (fp32 phase) and 409 at 0.6 m (fp64 phase accumulation, north_star item 4)."""
    g = {0: ([2e-4, 3e-4, 1.8e-3, 1.9e-3], [0, 10e-3, 10e-3, 0])}
    rf = ([0.0], [1e-4], [(math.pi / 2) / (W.GAMMA * 1e-4)], [0.0])
    s = seq(g=g, rf=rf, adc=3e-4 + (np.arange(300) + 0.5) * 5e-6, t_end=2e-3, dt_rf_max=1e-5)
    for kw, phase, turns in ((dict(), B.PHASE_FP32, (165, 180)), (dict(max_extent_m=0.6), B.PHASE_FP64, (400, 420)),
                             (dict(max_offres_hz=150e3), B.PHASE_FP64, (445, 465)),
                             (dict(max_extent_m=0.6, phase_mode="fp32"), B.PHASE_FP32, (400, 420))):
        h = B.bloch_plan_create(s, **kw)
        info = B.bloch_plan_get_info(h)
        B.bloch_plan_destroy(h)
        assert info["phase_mode"] == phase, kw
        assert turns[0] < info["worst_turns"] < turns[1], (kw, info["worst_turns"])
        assert info["max_extent_m"] == kw.get("max_extent_m", 0.25)
        assert info["max_offres_hz"] == kw.get("max_offres_hz", 1000.0) and info["max_speed_mps"] == 1.0
        assert info["phase_mode_requested"] == B._PHASE[kw.get("phase_mode", "auto")]
    # beyond the fp64 path's 2^19-turn fixed-point fraction: rejected at creation, not silently wrong
    with pytest.raises(B.BlochError) as e:
        B.bloch_plan_create(s, max_extent_m=1000.0)
    assert e.value.code == -10   # BLOCH_ERANGE
    with pytest.raises(B.BlochError) as e:
        B.bloch_plan_create(s, max_extent_m=float("nan"))
    assert e.value.code == -1


def test_waveform_motion_plan_merges_the_vertices_like_the_oracle(B, oracle_mod):
    """BLOCH_MOTION_WAVEFORM: the vertices of u(t) inside the sequence are points of the planner's grid exactly as they
    are of the oracle's, on top of the dt_max refinement; vertices outside [0, t_end] only shape u."""
    w = W.small("1")
    wf = (np.array([-1e-3, 1.234e-4, 3.3e-4, 9.871e-4, w.seq.t_end + 1e-3]), np.array([0.0, 0.5, 1.0, -1.0, 0.0]))
    for dt_max in (0.0, 3e-5):
        h = B.bloch_plan_create(w.seq, motion="waveform", waveform=wf, dt_max=dt_max)
        info = B.bloch_plan_get_info(h)
        B.bloch_plan_destroy(h)
        t, _, rf, _ = oracle_mod.grid(w.seq, dt_max=dt_max, waveform=wf)
        assert info["n_intervals"] == len(t) - 1 and info["n_rf_steps"] == int(rf.sum()) and info["motion_mode"] == 2
    h = B.bloch_plan_create(w.seq, motion="linear", dt_max=3e-5)
    assert B.bloch_plan_get_info(h)["n_intervals"] < info["n_intervals"]     # the inner vertices added points
    B.bloch_plan_destroy(h)


def test_adc_samples_inside_an_rf_run_cut_it_with_empty_precession_blocks(B, oracle_mod):
    """Reading G7: an ADC sample with RF on both sides is Mxy as it stands at that step boundary (what the oracle records).
    The planner serves it with an EMPTY precession block that cuts the RF run; also at t = 0 and at t_end."""
    n = 40
    rf = (np.arange(n) * 1e-5, np.full(n, 1e-5), np.full(n, 2e-6), np.zeros(n))
    s = seq(rf=rf, adc=[0.0, 5e-5, 1.3e-4, 1.35e-4, 4e-4], t_end=4e-4, dt_rf_max=1e-5)   # the RF run is the whole sequence
    h = B.bloch_plan_create(s)
    info = B.bloch_plan_get_info(h)
    B.bloch_plan_destroy(h)
    t, _, rfm, adc = oracle_mod.grid(s)
    assert info["n_intervals"] == len(t) - 1 and info["n_rf_steps"] == int(rfm.sum())
    # 1.35e-4 is not an RF sample edge: it becomes a grid point that splits one RF sample into two steps
    assert info["n_rf_steps"] == n + 1
    assert info["n_adc"] == 5 and info["n_rf_blocks"] == 4 and info["n_blocks"] == 9 and info["max_block_adc"] == 1
    assert info["n_eval_points"] == info["n_adc"] + (info["n_blocks"] - info["n_rf_blocks"])
