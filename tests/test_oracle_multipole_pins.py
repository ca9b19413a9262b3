"""Pins of the oracle's cell multipoles (Eq. 4): expected values come from the
equation evaluated another way (numpy monomials in a different association), closed forms and
invariants -- never from the oracle itself."""
import numpy as np

import oracle

CPD = 5
CELL = 1.0 / CPD


def _offsets(pos, cpd):
    t = pos.astype(np.float64) * cpd
    return (t - np.floor(t) - 0.5) / cpd, (np.floor(t).astype(int) % cpd)


def test_M1_basis_size_and_index_order():
    """(p+3)(p+2)(p+1)/6 values: 165 at p = 8; reduced basis (p+1)^2 = 81 is 'about
    half'.  Index order = the pseudo-code's nesting: a outer, then b, then c."""
    for p in (0, 1, 2, 8):
        idx = oracle.multipole_index(p)
        assert len(idx) == (p + 3) * (p + 2) * (p + 1) // 6
        assert all(a + b + c <= p for a, b, c in idx) and len(set(idx)) == len(idx)
    assert oracle.multipole_index(1) == [(0, 0, 0), (0, 0, 1), (0, 1, 0), (1, 0, 0)]
    assert len(oracle.multipole_index(8)) == 165 and 81 / 165 < 0.5


def test_M2_single_particle_is_its_monomials():
    pos = np.array([[0.31, 0.52, 0.77]], dtype=np.float32)
    off, c = _offsets(pos, CPD)
    M = oracle.multipoles(pos, CPD, 8)
    key = (c[0, 0] * CPD + c[0, 1]) * CPD + c[0, 2]
    x, y, z = off[0]
    want = np.array([x ** a * y ** b * z ** k for a, b, k in oracle.multipole_index(8)])
    assert np.allclose(M[key], want, rtol=1e-13, atol=0)
    assert np.count_nonzero(np.delete(M, key, axis=0)) == 0


def test_M3_low_orders_are_count_dipole_and_second_moments():
    rng = np.random.default_rng(7)
    pos = rng.random((3000, 3)).astype(np.float32)
    off, c = _offsets(pos, CPD)
    key = (c[:, 0] * CPD + c[:, 1]) * CPD + c[:, 2]
    M = oracle.multipoles(pos, CPD, 2)
    idx = oracle.multipole_index(2)
    assert np.array_equal(M[:, idx.index((0, 0, 0))], np.bincount(key, minlength=CPD ** 3).astype(float))
    for k, t in enumerate([(1, 0, 0), (0, 1, 0), (0, 0, 1)]):
        assert np.allclose(M[:, idx.index(t)], np.bincount(key, weights=off[:, k], minlength=CPD ** 3), rtol=1e-12, atol=1e-15)
    assert np.allclose(M[:, idx.index((1, 1, 0))], np.bincount(key, weights=off[:, 0] * off[:, 1], minlength=CPD ** 3), rtol=1e-12, atol=1e-16)
    assert np.allclose(M[:, idx.index((0, 0, 2))], np.bincount(key, weights=off[:, 2] ** 2, minlength=CPD ** 3), rtol=1e-12, atol=1e-16)


def test_M4_brute_force_all_terms_order_8():
    rng = np.random.default_rng(8)
    pos = rng.random((1500, 3)).astype(np.float32)
    off, c = _offsets(pos, CPD)
    key = (c[:, 0] * CPD + c[:, 1]) * CPD + c[:, 2]
    M = oracle.multipoles(pos, CPD, 8)
    for col, (a, b, k) in enumerate(oracle.multipole_index(8)):
        w = np.power(off[:, 0], a) * np.power(off[:, 1], b) * np.power(off[:, 2], k)
        ref = np.bincount(key, weights=w, minlength=CPD ** 3)
        scale = np.bincount(key, weights=np.abs(w), minlength=CPD ** 3)
        assert np.all(np.abs(M[:, col] - ref) <= 1e-13 * scale + 1e-300), (a, b, k)


def test_M5_mirror_symmetric_cell_has_no_odd_moments_and_bounds():
    """particles placed in +/- pairs about a cell centre: every moment of odd total order vanishes
    (to the rounding of a double sum); |M^{abc}| <= n (cell/2)^(a+b+c).  box = CPD so that the cell
    centre and the offsets (multiples of 2^-20) are exact in float32."""
    rng = np.random.default_rng(9)
    d = np.round((rng.random((40, 3)) - 0.5) * 0.8 * 2 ** 20) / 2 ** 20
    centre = np.array([2, 3, 1]) + 0.5
    pos = np.concatenate([centre + d, centre - d])
    pos32 = pos.astype(np.float32)
    assert np.array_equal(pos32.astype(np.float64), pos)
    M = oracle.multipoles(pos32, CPD, 8, box=float(CPD))
    key = (2 * CPD + 3) * CPD + 1
    for col, (a, b, k) in enumerate(oracle.multipole_index(8)):
        bound = 80 * 0.5 ** (a + b + k)
        if (a + b + k) % 2 == 1:
            assert abs(M[key, col]) <= 1e-14 * bound, (a, b, k)
        assert abs(M[key, col]) <= bound * (1 + 1e-12)
    assert M[key, 0] == 80.0


def test_M6_whole_cell_translation_and_input_order():
    """box = CPD (cell size 1): shifting by whole cells permutes the cells' multipoles exactly;
    permuting the input changes nothing beyond the order of a double sum."""
    rng = np.random.default_rng(10)
    pos = (np.floor(rng.random((2000, 3)) * CPD * 2 ** 16) / 2 ** 16).astype(np.float32)    # exact in float32, also after the shift
    M0 = oracle.multipoles(pos, CPD, 6, box=float(CPD))
    shifted = np.mod(pos.astype(np.float64) + np.array([1.0, 2.0, 3.0]), CPD).astype(np.float32)
    M1 = oracle.multipoles(shifted, CPD, 6, box=float(CPD)).reshape(CPD, CPD, CPD, -1)
    M1 = np.roll(M1, shift=(-1, -2, -3), axis=(0, 1, 2)).reshape(CPD ** 3, -1)
    assert np.array_equal(M0, M1)
    perm = rng.permutation(2000)
    M2 = oracle.multipoles(pos[perm], CPD, 6, box=float(CPD))
    assert np.allclose(M0, M2, rtol=1e-12, atol=1e-14)
