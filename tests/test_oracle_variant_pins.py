"""Pins of the oracle's build-time variants (``oracle.accel_variant``): Plummer softening
(Eq. 2) and the FoF-scale density estimate.  Same idea as
tests/test_oracle_pins.py: each expected value comes from the paper's formula evaluated by
hand, a closed form, an invariant, or a brute force over all pairs -- never from the oracle.
"""
import math

import numpy as np

import oracle

CPD, R = 7, 2
CELL = 1.0 / CPD


def _two(sep, axis=0, base=(0.5, 0.5, 0.5)):
    p = np.array([base, base], dtype=np.float64)
    p[1, axis] += sep
    return p.astype(np.float32)


# ---------------------------------------------------------------- Plummer, Eq. 2
def test_V1_plummer_two_particle_closed_form():
    """F = r/(r^2+eps^2)^(3/2).  Hand values of g(x) = x/(1+x^2)^(3/2), x = r/eps:
    g(1) = 2^-1.5, g(2) = 2/5^1.5, g(0.5) = 0.5/1.25^1.5; maximum 2/(3 sqrt 3) at x = 1/sqrt 2."""
    eps = 0.01
    hand = {0.5: 0.5 / 1.25 ** 1.5, 1.0: 2.0 ** -1.5, 2.0: 2.0 / 5.0 ** 1.5, 1.0 / math.sqrt(2.0): 2.0 / (3.0 * math.sqrt(3.0))}
    for x, g in hand.items():
        pos = _two(x * eps)
        d = float(pos[1, 0]) - float(pos[0, 0])          # the float32 separation the oracle sees
        xx = d / eps
        expect = xx / (1.0 + xx * xx) ** 1.5
        assert abs(expect - g) < 3e-5 * g + 1e-4 * abs(1 - 2 * x * x)  # float32 input rounding only (flat at the maximum)
        acc, _, pairs = oracle.accel_variant(pos, CPD, R, eps, gm=1.0, law="plummer")
        assert pairs == 2
        assert np.allclose(acc[0], [expect / eps ** 2, 0, 0], rtol=1e-12, atol=0)
        assert np.allclose(acc[1], -acc[0], rtol=0, atol=0)


def test_V2_plummer_large_r_is_newtonian_and_below_it():
    """Eq. 2 converges to r^-2 from below, 'only converging quadratically':
    1 - F r^2 = 1.5 (eps/r)^2 + O((eps/r)^4)."""
    eps = 1e-3
    pos = _two(0.1)
    d = float(pos[1, 0]) - float(pos[0, 0])
    acc, _, _ = oracle.accel_variant(pos, CPD, R, eps, gm=1.0, law="plummer")
    defect = 1.0 - acc[0, 0] * d * d
    assert 0 < defect
    assert abs(defect - 1.5 * (eps / d) ** 2) < 3 * (eps / d) ** 4


def test_V3_plummer_brute_force_all_pairs_masked():
    """all-pairs loop with particle minimum image, masked to near-field cell pairs (CPD >= 2R+2)."""
    rng = np.random.default_rng(5)
    N, eps = 600, 0.02
    pos = rng.random((N, 3)).astype(np.float32)
    acc, _, pairs = oracle.accel_variant(pos, CPD, R, eps, gm=1.0 / N, law="plummer")
    x = pos.astype(np.float64)
    cell = np.floor(x * CPD).astype(int) % CPD
    ref = np.zeros((N, 3))
    npairs = 0
    for i in range(N):
        d = x - x[i]
        d -= np.round(d)
        dc = (cell - cell[i] + CPD // 2) % CPD - CPD // 2
        m = (np.abs(dc) <= R).all(axis=1)
        m[i] = False
        npairs += int(m.sum())
        s2 = (d[m] ** 2).sum(axis=1) + eps * eps
        ref[i] = (d[m] / s2[:, None] ** 1.5).sum(axis=0) / N
    assert pairs == npairs
    rms = np.sqrt((ref ** 2).sum(axis=1).mean())
    assert np.abs(acc - ref).max() < 1e-12 * rms


def test_V4_plummer_and_spline_agree_far_from_the_softening():
    """both laws are Newtonian to O((eps/r)^2) once r >> eps; momentum sum vanishes for both."""
    rng = np.random.default_rng(2)
    pos = rng.random((400, 3)).astype(np.float32)
    eps = 1e-6
    a0, _, _ = oracle.accel_variant(pos, CPD, R, eps, law="spline")
    a1, _, _ = oracle.accel_variant(pos, CPD, R, eps, law="plummer")
    assert np.abs(a0 - a1).max() < 1e-6 * np.abs(a0).max()
    assert np.abs(a1.sum(axis=0)).max() < 1e-13 * np.abs(a1).sum()
    b0, _ = oracle.accel(pos, CPD, R, eps)
    assert np.array_equal(a0, b0)            # law="spline" is the main oracle's arithmetic, term for term


# ---------------------------------------------------------------- density
def test_W1_density_two_particles():
    """b^2 - r^2 for r < b, nothing beyond b, the particle itself is not counted (reading D1)."""
    b = 0.03
    for sep in (0.01, 0.02, 0.029, 0.031, 0.1):
        pos = _two(sep, axis=1)
        d = float(pos[1, 1]) - float(pos[0, 1])
        _, dens, _ = oracle.accel_variant(pos, CPD, R, 1e-3, density_b=b)
        expect = b * b - d * d if d < b else 0.0
        assert np.allclose(dens, [expect, expect], rtol=1e-12, atol=1e-18)
    _, dens, _ = oracle.accel_variant(np.array([[0.3, 0.3, 0.3]], dtype=np.float32), CPD, R, 1e-3, density_b=b)
    assert dens[0] == 0.0


def test_W2_density_coincident_particles_count_b2():
    pos = np.array([[0.4, 0.4, 0.4]] * 3, dtype=np.float32)
    _, dens, _ = oracle.accel_variant(pos, CPD, R, 1e-3, density_b=0.05)
    assert np.allclose(dens, 2 * 0.05 ** 2, rtol=1e-15)          # reading D2


def test_W3_density_simple_cubic_lattice_shells():
    """one particle per cell on a cubic lattice of spacing a = cell: 6 neighbours at a, 12 at
    sqrt2 a, 8 at sqrt3 a -> closed-form shell sums for b between the shell radii."""
    g = (np.arange(CPD) + 0.5) / CPD
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3).astype(np.float32)
    a = CELL
    for b, shells in ((1.2 * a, [(6, 1.0)]), (1.5 * a, [(6, 1.0), (12, 2.0)]), (1.9 * a, [(6, 1.0), (12, 2.0), (8, 3.0)])):
        expect = sum(n * (b * b - k * a * a) for n, k in shells)
        _, dens, _ = oracle.accel_variant(pos, CPD, R, 1e-3, density_b=b)
        assert np.allclose(dens, expect, rtol=2e-6)               # float32 lattice coordinates


def test_W4_density_brute_force_and_wrap():
    rng = np.random.default_rng(11)
    N, b = 900, 0.9 * CELL
    pos = rng.random((N, 3)).astype(np.float32)
    _, dens, _ = oracle.accel_variant(pos, CPD, R, 1e-3, density_b=b)
    x = pos.astype(np.float64)
    ref = np.zeros(N)
    for i in range(N):
        d = x - x[i]
        d -= np.round(d)                                            # b < cell <= R cells: every r < b pair is a near-field pair
        r2 = (d ** 2).sum(axis=1)
        m = r2 < b * b
        m[i] = False
        ref[i] = (b * b - r2[m]).sum()
    assert np.abs(dens - ref).max() < 1e-12 * ref.max()
    # across the periodic boundary
    pos2 = np.array([[0.005, 0.5, 0.5], [0.995, 0.5, 0.5]], dtype=np.float32)
    _, d2, _ = oracle.accel_variant(pos2, CPD, R, 1e-3, density_b=0.02)
    sep = 1.0 - (float(pos2[1, 0]) - float(pos2[0, 0]))
    assert np.allclose(d2, 0.02 ** 2 - sep ** 2, rtol=1e-9)


def test_W5_density_mean_of_a_uniform_field():
    """<dens> = n * integral_0^b (b^2 - r^2) 4 pi r^2 dr = n (8 pi / 15) b^5 for a Poisson field."""
    rng = np.random.default_rng(3)
    N, b = 40000, 0.5 * CELL
    pos = rng.random((N, 3)).astype(np.float32)
    _, dens, _ = oracle.accel_variant(pos, CPD, R, 1e-3, density_b=b)
    expect = N * (8.0 * math.pi / 15.0) * b ** 5
    assert abs(dens.mean() - expect) < 0.03 * expect


def test_W6_density_does_not_change_the_force():
    rng = np.random.default_rng(4)
    pos = rng.random((500, 3)).astype(np.float32)
    a0, _, p0 = oracle.accel_variant(pos, CPD, R, 0.01)
    a1, d1, p1 = oracle.accel_variant(pos, CPD, R, 0.01, density_b=0.04)
    assert np.array_equal(a0, a1) and p0 == p1 and d1 is not None


# ---------------------------------------------------------------- no softening
def test_N1_newton_two_particle_inverse_square():
    """'Newtonian gravity, or a softened form thereof': |a| = gm / r^2 at every
    separation, however small, attractive, a1 = -a2; along an oblique direction too."""
    for sep in (1e-6, 1e-4, 0.003, 0.05, 0.2):
        pos = _two(sep)
        d = float(pos[1, 0]) - float(pos[0, 0])
        acc, _, pairs = oracle.accel_variant(pos, CPD, R, 0.01, gm=2.5, law="newton")
        assert pairs == 2
        assert np.allclose(acc[0], [2.5 / d ** 2, 0, 0], rtol=1e-13, atol=0)
        assert np.array_equal(acc[1], -acc[0])
    p = np.array([[0.5, 0.5, 0.5], [0.5 + 0.02, 0.5 - 0.01, 0.5 + 0.02]], dtype=np.float32)
    dv = p[1].astype(np.float64) - p[0].astype(np.float64)
    acc, _, _ = oracle.accel_variant(p, CPD, R, 0.01, gm=1.0, law="newton")
    assert np.allclose(acc[0], dv / np.linalg.norm(dv) ** 3, rtol=1e-12)


def test_N2_newton_ignores_eps_and_is_the_limit_of_both_softened_laws():
    """eps_p does not enter; Eq. 3 equals it exactly once every pair has r >= eps_s (compact
    support); Eq. 2 approaches it as 1.5 (eps/r)^2."""
    rng = np.random.default_rng(12)
    pos = rng.random((300, 3)).astype(np.float32)
    a_n, _, p_n = oracle.accel_variant(pos, CPD, R, 0.01, law="newton")
    a_n2, _, _ = oracle.accel_variant(pos, CPD, R, 3.0, law="newton")
    assert np.array_equal(a_n, a_n2)
    x = pos.astype(np.float64)
    dmin = min(np.sqrt((((x - x[i]) - np.round(x - x[i])) ** 2).sum(1))[np.arange(300) != i].min() for i in range(300))
    eps = 0.4 * dmin / 2.16                                   # eps_s = 2.16 eps < every separation
    a_s, _, p_s = oracle.accel_variant(pos, CPD, R, eps, law="spline")
    assert p_s == p_n
    assert np.abs(a_s - a_n).max() <= 1e-13 * np.abs(a_n).max()
    a_p, _, _ = oracle.accel_variant(pos, CPD, R, 1e-7, law="plummer")
    assert np.abs(a_p - a_n).max() <= 1e-6 * np.abs(a_n).max()
    assert np.abs(a_n.sum(axis=0)).max() < 1e-13 * np.abs(a_n).sum()        # momentum


def test_N3_newton_brute_force_all_pairs_masked():
    rng = np.random.default_rng(6)
    N = 500
    pos = rng.random((N, 3)).astype(np.float32)
    acc, _, pairs = oracle.accel_variant(pos, CPD, R, 0.02, gm=1.0 / N, law="newton")
    x = pos.astype(np.float64)
    cell = np.floor(x * CPD).astype(int) % CPD
    ref = np.zeros((N, 3))
    npairs = 0
    for i in range(N):
        d = x - x[i]
        d -= np.round(d)
        dc = (cell - cell[i] + CPD // 2) % CPD - CPD // 2
        m = (np.abs(dc) <= R).all(axis=1)
        m[i] = False
        npairs += int(m.sum())
        r2 = (d[m] ** 2).sum(axis=1)
        ref[i] = (d[m] / r2[:, None] ** 1.5).sum(axis=0) / N
    assert pairs == npairs
    rms = np.sqrt((ref ** 2).sum(axis=1).mean())
    assert np.abs(acc - ref).max() < 1e-12 * rms


def test_N4_newton_coincident_particles_contribute_nothing():
    """reading N1: F(0) = 0 for a coincident pair, as for the softened laws (S4) -- no Inf/NaN."""
    pos = np.array([[0.3, 0.3, 0.3], [0.3, 0.3, 0.3], [0.35, 0.3, 0.3]], dtype=np.float32)
    acc, _, pairs = oracle.accel_variant(pos, CPD, R, 0.01, gm=1.0, law="newton")
    d = float(pos[2, 0]) - float(pos[0, 0])
    assert pairs == 6 and np.isfinite(acc).all()
    assert np.allclose(acc[0], [1 / d ** 2, 0, 0], rtol=1e-13) and np.array_equal(acc[0], acc[1])
    assert np.allclose(acc[2], [-2 / d ** 2, 0, 0], rtol=1e-13)
