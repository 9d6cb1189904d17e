"""Tiny hand-built sequences/phantoms for the pins (test helper; no solver arithmetic)."""
import numpy as np

from paper_2301_02702_b200.workloads import Phantom, Sequence

Z = np.zeros(0)


def phantom(x=0.0, y=0.0, z=0.0, M0=1.0, T1=1e30, T2=1e30, dw=0.0):
    arrs = np.broadcast_arrays(*[np.atleast_1d(np.asarray(a, dtype=np.float64)) for a in (x, y, z, M0, T1, T2, dw)])
    return Phantom(*[np.ascontiguousarray(a, dtype=np.float64) for a in arrs])


def seq(g=None, rf=None, adc=(), t_end=1.0, dt_rf_max=1e-6):
    """g: dict axis-> (times, values); rf: (t, dt, re, im) arrays."""
    g = g or {}
    g_t = [np.asarray(g.get(a, (Z, Z))[0], dtype=np.float64) for a in range(3)]
    g_v = [np.asarray(g.get(a, (Z, Z))[1], dtype=np.float64) for a in range(3)]
    if rf is None:
        rf = (Z, Z, Z, Z)
    rf = [np.atleast_1d(np.asarray(a, dtype=np.float64)) for a in rf]
    return Sequence(g_t, g_v, rf[0], rf[1], rf[2], rf[3], np.atleast_1d(np.asarray(adc, dtype=np.float64)),
                    float(t_end), float(dt_rf_max))
