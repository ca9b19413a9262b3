"""Pins of the oracle's Taylor evaluation (reading F1 of DESIGN.md): closed forms
for low-order potentials, a numerical gradient of the polynomial for random coefficients, and the
independence of cells."""
import numpy as np

import oracle

CPD = 4


def _offsets(pos, cpd):
    t = pos.astype(np.float64) * cpd
    c = np.floor(t).astype(int) % cpd
    return (t - np.floor(t) - 0.5) / cpd, (c[:, 0] * cpd + c[:, 1]) * cpd + c[:, 2]


def _phi(T, idx, x, y, z):
    return sum(t * x ** a * y ** b * z ** c for t, (a, b, c) in zip(T, idx))


def test_F1_uniform_field_and_harmonic_potential():
    rng = np.random.default_rng(0)
    pos = rng.random((500, 3)).astype(np.float32)
    off, key = _offsets(pos, CPD)
    idx = oracle.multipole_index(2)
    T = np.zeros((CPD ** 3, len(idx)))
    T[:, idx.index((1, 0, 0))] = 3.0           # phi = 3x - 2z: a = (-3, 0, 2) everywhere
    T[:, idx.index((0, 0, 1))] = -2.0
    acc = oracle.taylor_accel(pos, T, CPD, 2)
    assert np.allclose(acc, [-3.0, 0.0, 2.0], rtol=0, atol=1e-15)
    T[:] = 0
    k = np.arange(CPD ** 3) + 1.0              # phi = k/2 r^2 with a different k per cell: a = -k * offset
    for t in ((2, 0, 0), (0, 2, 0), (0, 0, 2)):
        T[:, idx.index(t)] = 0.5 * k
    acc = oracle.taylor_accel(pos, T, CPD, 2)
    assert np.allclose(acc, -k[key][:, None] * off, rtol=1e-14, atol=1e-18)


def test_F2_single_monomials_closed_form():
    pos = np.array([[0.30, 0.55, 0.80]], dtype=np.float32)
    off, key = _offsets(pos, CPD)
    x, y, z = off[0]
    idx = oracle.multipole_index(8)
    for (a, b, c) in [(8, 0, 0), (0, 0, 8), (3, 2, 1), (1, 1, 1), (0, 4, 4), (2, 0, 5), (0, 0, 0)]:
        T = np.zeros((CPD ** 3, len(idx)))
        T[key[0], idx.index((a, b, c))] = 1.7
        acc = oracle.taylor_accel(pos, T, CPD, 8)[0]
        want = -1.7 * np.array([a * x ** max(a - 1, 0) * y ** b * z ** c if a else 0.0,
                                b * x ** a * y ** max(b - 1, 0) * z ** c if b else 0.0,
                                c * x ** a * y ** b * z ** max(c - 1, 0) if c else 0.0])
        assert np.allclose(acc, want, rtol=1e-13, atol=1e-300), (a, b, c)


def test_F3_random_coefficients_against_a_numerical_gradient():
    rng = np.random.default_rng(3)
    pos = rng.random((60, 3)).astype(np.float32)
    off, key = _offsets(pos, CPD)
    idx = oracle.multipole_index(8)
    T = rng.normal(size=(CPD ** 3, len(idx))) * np.array([CPD ** (a + b + c) for a, b, c in idx])    # every order matters
    acc = oracle.taylor_accel(pos, T, CPD, 8)
    h = 1e-6 / CPD
    for i in range(60):
        x, y, z = off[i]
        t = T[key[i]]
        g = np.array([(_phi(t, idx, x + h, y, z) - _phi(t, idx, x - h, y, z)) / (2 * h),
                      (_phi(t, idx, x, y + h, z) - _phi(t, idx, x, y - h, z)) / (2 * h),
                      (_phi(t, idx, x, y, z + h) - _phi(t, idx, x, y, z - h)) / (2 * h)])
        assert np.allclose(acc[i], -g, rtol=2e-7, atol=1e-7 * np.abs(g).max())


def test_F4_cells_are_independent_and_input_order_is_kept():
    rng = np.random.default_rng(4)
    pos = rng.random((300, 3)).astype(np.float32)
    _, key = _offsets(pos, CPD)
    idx = oracle.multipole_index(4)
    T = rng.normal(size=(CPD ** 3, len(idx)))
    a0 = oracle.taylor_accel(pos, T, CPD, 4)
    T2 = T.copy()
    T2[5] += 1.0                                   # changing one cell's coefficients moves only its particles
    a1 = oracle.taylor_accel(pos, T2, CPD, 4)
    assert np.array_equal(a0[key != 5], a1[key != 5]) and (key == 5).any() and not np.array_equal(a0[key == 5], a1[key == 5])
    perm = rng.permutation(300)
    assert np.array_equal(oracle.taylor_accel(pos[perm], T, CPD, 4), a0[perm])
