"""Files for the objects that cross the boundary (PAPER.md:93 Fig 1, :99-101): the library's OWN text container for
scanner + sequence and for the raw signal -- not Pulseq, not ISMRMRD.  Pinned by round trips: the
arrays come back bit for bit, and a plan built from the file has bitwise the tables of a plan built from the arrays."""
import os

import numpy as np
import pytest

from paper_2301_02702_b200 import build as bl
from paper_2301_02702_b200 import workloads as W


@pytest.fixture(scope="module")
def B():
    bl.build()
    from paper_2301_02702_b200 import bloch
    return bloch


@pytest.mark.parametrize("name", ["1", "2", "3", "4", "5", "5b"])
def test_sequence_file_round_trip_is_bit_exact_and_gives_the_same_plan(B, tmp_path, name):
    w = W.small(name)
    path = str(tmp_path / f"config{name}.bseq")
    B.bloch_sequence_write(path, w.seq, gamma=W.GAMMA, B0=1.5, G_max=60e-3, S_max=500.0)
    scanner, seq = B.bloch_sequence_read(path)
    assert scanner == dict(gamma=W.GAMMA, B0=1.5, G_max=60e-3, S_max=500.0)
    for a in range(3):
        assert np.array_equal(seq.g_t[a], w.seq.g_t[a]) and np.array_equal(seq.g_v[a], w.seq.g_v[a])
    for k in ("rf_t", "rf_dt", "rf_re", "rf_im", "adc_t"):
        assert np.array_equal(getattr(seq, k), np.asarray(getattr(w.seq, k), dtype=np.float64)), k
    assert seq.t_end == w.seq.t_end
    kw = dict(dt_rf_max=w.seq.dt_rf_max, phase_mode=w.phase_mode, output_mode=w.output_mode)
    h0 = B.bloch_plan_create(w.seq, **kw)
    h1 = B.bloch_plan_create(seq, gamma=scanner["gamma"], **kw)
    try:
        assert B.bloch_plan_get_info(h0) == B.bloch_plan_get_info(h1)
        t0, t1 = B.bloch_plan_host_tables(h0), B.bloch_plan_host_tables(h1)
        assert len(t0) == B.bloch_plan_get_info(h0)["table_bytes"] and t0 == t1, "plan tables differ after the round trip"
    finally:
        B.bloch_plan_destroy(h0)
        B.bloch_plan_destroy(h1)


def test_signal_file_round_trip(B, tmp_path):
    rng = np.random.default_rng(5)
    for shape in ((37,), (3, 11), (1, 0)):
        sig = (rng.normal(size=shape) + 1j * rng.normal(size=shape)).astype(np.complex64)
        n_adc = shape[-1]
        t = np.sort(rng.uniform(0, 1, n_adc))
        path = str(tmp_path / "s.bsig")
        B.bloch_signal_write(path, sig, adc_t=t)
        got, tt = B.bloch_signal_read(path)
        assert np.array_equal(got.reshape(sig.shape).view(np.float32), sig.view(np.float32)) and np.array_equal(tt, t)
        B.bloch_signal_write(path, sig)                      # without sample times
        got, _ = B.bloch_signal_read(path)
        assert np.array_equal(got.reshape(sig.shape).view(np.float32), sig.view(np.float32))


def test_file_errors(B, tmp_path):
    with pytest.raises(B.BlochError) as e:
        B.bloch_sequence_read(str(tmp_path / "missing.bseq"))
    assert e.value.code == -1
    p = tmp_path / "other.seq"
    p.write_text("# Pulseq sequence file\n[VERSION]\nmajor 1\n")          # another format's file is refused, not guessed at
    with pytest.raises(B.BlochError) as e:
        B.bloch_sequence_read(str(p))
    assert e.value.code == -1 and "own format" in str(e.value)
    w = W.small("1")
    good = tmp_path / "good.bseq"
    B.bloch_sequence_write(str(good), w.seq)
    text = good.read_text()
    (tmp_path / "cut.bseq").write_text(text[: len(text) // 2])             # truncated
    with pytest.raises(B.BlochError):
        B.bloch_sequence_read(str(tmp_path / "cut.bseq"))
    (tmp_path / "bad.bsig").write_text("bloch-signal 2\n")
    with pytest.raises(B.BlochError):
        B.bloch_signal_read(str(tmp_path / "bad.bsig"))
    assert os.path.exists(str(good))
