"""Pins of the oracle's multi-coil receive (SURVEY.md 8(f) f2 "per-coil weights"; reading C1: S_c(t) = sum_i C_c(x_i)
Mxy_i(t), the paper itself has no coils yet).  Closed form with complex weights (a conjugated or
transposed weight matrix fails it), the degenerate weights, and a partition of unity."""
import math

import numpy as np

from seqtools import phantom, seq

GAMMA = 2.0 * math.pi * 42.58e6


def test_c1_weighted_free_precession_closed_form(oracle_mod):
    # after an ideal state (Mxy = i M0) each spin's signal is i M0 exp(-t/T2) exp(-i(gamma G x + dw) t)  (P1, P2)
    x = np.array([0.01, -0.03, 0.05]); dw = np.array([30.0, -80.0, 10.0]); T2 = np.array([0.05, 0.1, 0.2])
    M0 = np.array([1.0, 0.7, 0.4])
    ph = phantom(x=x, M0=M0, T2=T2, T1=1e30, dw=dw)
    Gx = 2e-3
    adc = np.array([0.0, 1e-3, 3.3e-3, 9e-3])
    s = seq(g={0: ([0.0, 1e-2], [Gx, Gx])}, adc=adc, t_end=1e-2)
    W = np.array([[1 + 2j, -0.5j, 0.25], [0.3 - 1j, 2.0, -1 + 1j]])
    st = (1j * M0, np.zeros(3))
    got = oracle_mod.simulate(ph, s, state=st, coils=W)
    per = (1j * M0)[:, None] * np.exp(-adc[None, :] / T2[:, None]) * \
        np.exp(-1j * (GAMMA * Gx * x[:, None] + dw[:, None]) * adc[None, :])
    want = np.stack([(W[c][:, None] * per).sum(axis=0) for c in range(2)])
    assert got.shape == (2, 4)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-12)
    assert np.abs(got - np.conj(W) @ per).max() > 0.1 and np.abs(got[0] - got[1]).max() > 0.1


def test_c1_degenerate_weights_and_partition_of_unity(oracle_mod):
    rng = np.random.default_rng(3)
    n = 40
    ph = phantom(x=rng.uniform(-.1, .1, n), y=rng.uniform(-.1, .1, n), M0=rng.uniform(.5, 1, n),
                 T1=rng.uniform(.3, 2, n), T2=rng.uniform(.03, .3, n), dw=rng.uniform(-200, 200, n))
    rf = (np.arange(50) * 1e-5, np.full(50, 1e-5), np.full(50, (math.pi / 3) / (GAMMA * 5e-4)), np.zeros(50))
    s = seq(g={0: ([6e-4, 7e-4, 3e-3], [0, 5e-3, 5e-3])}, rf=rf, adc=8e-4 + np.arange(64) * 2e-5, t_end=3e-3,
            dt_rf_max=1e-5)
    plain = oracle_mod.simulate(ph, s)
    ones = oracle_mod.simulate(ph, s, coils=np.ones((1, n)))
    np.testing.assert_allclose(ones[0], plain, rtol=0, atol=1e-13)                  # one uniform coil = no coil
    c = 0.7 * np.exp(1j * 1.1)
    np.testing.assert_allclose(oracle_mod.simulate(ph, s, coils=np.full((1, n), c))[0], c * plain, rtol=0, atol=1e-13)
    # smooth sensitivities that add up to one everywhere: the coil signals add up to the plain signal
    a = 0.5 + 0.5 * np.tanh(ph.x / 0.03)
    W = np.stack([a * np.exp(1j * ph.y * 20), (1 - a) * np.exp(1j * ph.y * 20), 1 - np.exp(1j * ph.y * 20)])
    got = oracle_mod.simulate(ph, s, coils=W)
    np.testing.assert_allclose(got.sum(axis=0), plain, rtol=0, atol=1e-12)
    # a coil that sees one spin only returns that spin's own signal
    per = oracle_mod.simulate(ph, s, output_mode="per_spin")
    e = np.zeros((1, n)); e[0, 17] = 1.0
    np.testing.assert_allclose(oracle_mod.simulate(ph, s, coils=e)[0], per[17], rtol=0, atol=1e-15)
