"""Pins of the oracle's Kick/Drift (Table 1 :379-380) and of the particle part of the
time-step criterion, Eq. 1: closed forms of the leapfrog, the periodic wrap,
hand-built cells."""
import math

import numpy as np

import oracle


def test_K1_constant_acceleration_is_integrated_exactly_by_kdk():
    """KDK with constant a: half kick, drift, half kick gives x0 + v0 t + a t^2/2 and v0 + a t
    (second-order leapfrog is exact for a quadratic trajectory).  Values exact in float32."""
    p = np.array([[0.25, 0.5, 0.125]], dtype=np.float32)
    v = np.array([[0.125, -0.25, 0.0]], dtype=np.float32)
    a = np.array([[0.5, 0.25, -0.5]], dtype=np.float32)
    t = 0.25
    p1, v1 = oracle.kick_drift(p, v, a, t / 2, t)            # half kick + drift
    _, v2 = oracle.kick_drift(p1, v1, a, t / 2, 0.0)         # second half kick, no drift
    assert np.array_equal(p1, (p.astype(np.float64) + v * t + 0.5 * a * t * t).astype(np.float32))
    assert np.array_equal(v2, (v.astype(np.float64) + a * t).astype(np.float32))


def test_K2_periodic_wrap_and_fold():
    p = np.array([[0.95, 0.05, 0.5], [0.5, 0.5, 0.5]], dtype=np.float32)
    v = np.array([[1.0, -1.0, 0.0], [3.0, -3.0, 7.0]], dtype=np.float32)
    z = np.zeros_like(v)
    p1, v1 = oracle.kick_drift(p, v, z, 0.0, 0.1)
    assert np.array_equal(v1, v)
    want0 = np.array([0.95 + 0.1 - 1.0, 0.05 - 0.1 + 1.0, 0.5])
    assert np.allclose(p1[0], want0, atol=1e-7) and np.all((p1 >= 0) & (p1 < 1))
    p2, _ = oracle.kick_drift(p, v, z, 0.0, 1.0)              # several periods: 0.5 + 3 -> 0.5, 0.5 - 3 -> 0.5, 0.5 + 7 -> 0.5
    assert np.allclose(p2[1], [0.5, 0.5, 0.5], atol=1e-6)
    # a value that would round to box folds to 0
    tiny = np.array([[1e-9, 0.0, 0.0]], dtype=np.float32)
    p3, _ = oracle.kick_drift(tiny, np.array([[-1.0, 0, 0]], dtype=np.float32), np.zeros((1, 3), np.float32), 0.0, 2e-9)
    assert p3[0, 0] == 0.0 or 0.0 <= p3[0, 0] < 1.0
    assert p3[0, 0] != 1.0
    # other box sizes
    p4, _ = oracle.kick_drift(np.array([[4.5, 0.5, 2.0]], np.float32), np.array([[1.0, -1.0, 0.0]], np.float32),
                              np.zeros((1, 3), np.float32), 0.0, 1.0, box=5.0)
    assert np.allclose(p4[0], [0.5, 4.5, 2.0])


def test_K3_harmonic_oscillator_energy_stays_bounded():
    """leapfrog on a = -x (about the box centre): energy error O(dt^2), no drift over many periods."""
    x = np.array([[0.6, 0.5, 0.5]], dtype=np.float32)
    v = np.zeros((1, 3), dtype=np.float32)
    dt = 0.05
    e0 = 0.5 * 0.1 ** 2
    acc = lambda x: (-(x.astype(np.float64) - 0.5)).astype(np.float32)
    _, v = oracle.kick_drift(x, v, acc(x), dt / 2, 0.0)
    worst = 0.0
    for _ in range(2000):
        x, v = oracle.kick_drift(x, v, np.zeros_like(v), 0.0, dt)        # drift
        _, vh = oracle.kick_drift(x, v, acc(x), dt / 2, 0.0)             # synchronised velocity
        e = 0.5 * float((vh.astype(np.float64) ** 2).sum()) + 0.5 * float(((x.astype(np.float64) - 0.5) ** 2).sum())
        worst = max(worst, abs(e - e0) / e0)
        _, v = oracle.kick_drift(x, v, acc(x), dt, 0.0)                  # full kick to the next half step
    assert worst < 2e-3


def test_T1_timestep_ratio_hand_built_cells():
    """two occupied cells of a CPD 4 grid: cell A has v = (3,4,0),(0,0,0) -> v_rms = sqrt(25/2),
    a_max = 2; cell B has v = (1,0,0) and a = (0,0,10) -> ratio 0.1: the minimum.  Global:
    v_rms = sqrt(26/3), a_max = 10."""
    pos = np.array([[0.1, 0.1, 0.1], [0.12, 0.1, 0.1], [0.6, 0.6, 0.6]], dtype=np.float32)
    vel = np.array([[3, 4, 0], [0, 0, 0], [1, 0, 0]], dtype=np.float32)
    acc = np.array([[0, 2, 0], [1, 0, 0], [0, 0, 10]], dtype=np.float32)
    out = oracle.timestep_ratio(pos, vel, acc, 4)
    assert math.isclose(out[0], 0.1, rel_tol=1e-15)
    assert math.isclose(out[2], math.sqrt(26 / 3), rel_tol=1e-15) and out[3] == 10.0
    assert math.isclose(out[1], math.sqrt(26 / 3) / 10, rel_tol=1e-15)
    # not Galilean invariant: a bulk velocity raises v_rms
    out2 = oracle.timestep_ratio(pos, vel + np.float32(10), acc, 4)
    assert out2[0] > out[0] and out2[2] > out[2]


def test_T2_cells_without_acceleration_do_not_constrain_and_brute_force():
    rng = np.random.default_rng(1)
    N, cpd = 4000, 5
    pos = rng.random((N, 3)).astype(np.float32)
    vel = rng.normal(size=(N, 3)).astype(np.float32)
    acc = rng.normal(size=(N, 3)).astype(np.float32)
    cell, _ = oracle.bin_particles(pos, cpd)
    acc[cell == 7] = 0                                    # a cell with a_max = 0: skipped
    out = oracle.timestep_ratio(pos, vel, acc, cpd)
    best = np.inf
    for c in np.unique(cell):
        m = cell == c
        amax = np.sqrt((acc[m].astype(np.float64) ** 2).sum(1).max())
        if amax == 0:
            continue
        best = min(best, np.sqrt((vel[m].astype(np.float64) ** 2).sum(1).mean()) / amax)
    assert math.isclose(out[0], best, rel_tol=1e-13)
    assert math.isclose(out[2], np.sqrt((vel.astype(np.float64) ** 2).sum(1).mean()), rel_tol=1e-13)
    assert math.isclose(out[3], np.sqrt((acc.astype(np.float64) ** 2).sum(1).max()), rel_tol=1e-15)
    assert out[0] <= out[1]                               # the most conservative cell is below the global ratio
    none = oracle.timestep_ratio(pos, vel, np.zeros_like(acc), cpd)
    assert np.isinf(none[0]) and np.isinf(none[1]) and none[3] == 0.0
