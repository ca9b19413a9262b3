"""Pins for the CPU oracle (``oracle/nf_oracle.c``) against what the paper and the
mathematics fix -- none of them re-types the oracle's own loop.

P1  closed form of Eq. 3 for two particles, values in tests/golden
P2  cell-based (not distance-based) cutoff
P3  periodic wrap, PAPER.md:232
P4  one particle per cell => zero force (stencil inversion symmetry)
P5  momentum: sum_i a_i = 0 (symmetric neighbour relation, antisymmetric F)
P6  brute force: all pairs, particle minimum image, masked to wrapped cell delta <= R
P7  integer pair-count identity with a separable periodic box filter
P8  CPD = 2R+1 => every cell neighbours every cell once => plain all-pairs sum
P9  translation by whole cells
P10 input-order invariance
P11 eps_s = 2.16 eps_p "to match the small-scale Plummer force"
"""
import math
import os

import numpy as np
import pytest

from paper_2110_11392_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "eq3_force_table.txt")


def _two(oracle_mod, x1, x2, cpd, R, eps_p):
    pos = np.array([x1, x2], dtype=np.float32)
    acc, pairs = oracle_mod.accel(pos, cpd, R, eps_p, box=1.0, gm=1.0)
    return pos.astype(np.float64), acc, pairs


# ---------------------------------------------------------------- P1
def test_p1_two_particle_closed_form(oracle_mod):
    tab = np.loadtxt(GOLDEN)
    cpd, R = 8, 2                       # cell = 1/8 exactly representable
    eps_p = 0.02
    eps_s = 2.16 * eps_p
    for u, g in tab:
        r = u * eps_s
        # both particles inside one cell (cell [0.5,0.625)), separation along a skew direction
        n = np.array([2.0, -1.0, 2.0]) / 3.0
        x1 = np.array([0.52, 0.58, 0.53])
        x2 = x1 + r * n
        pos, acc, pairs = _two(oracle_mod, x1, x2, cpd, R, eps_p)
        d = pos[1] - pos[0]             # float32-rounded inputs are what the oracle sees
        rr = np.linalg.norm(d)
        uu = rr / eps_s
        g_exact = (10 * uu - 15 * uu ** 2 + 6 * uu ** 3) if uu < 1 else uu ** -2
        assert pairs == 2
        a1 = np.linalg.norm(acc[0]) * eps_s ** 2
        assert a1 == pytest.approx(g_exact, rel=1e-12)
        assert a1 == pytest.approx(g, rel=2e-5)          # golden value (float32 input rounding)
        assert np.allclose(acc[0], -acc[1], rtol=0, atol=1e-12 * abs(acc).max())
        # attractive: acceleration of particle 0 points towards particle 1
        assert np.dot(acc[0], d) > 0
        assert np.allclose(acc[0] / np.linalg.norm(acc[0]), d / rr, atol=1e-12)


def test_p1_force_maximum_and_c2_continuity(oracle_mod):
    eps_s = 0.3
    ustar = (30 - math.sqrt(180)) / 36
    g = lambda u: oracle_mod.force_factor(u * eps_s, eps_s) * (u * eps_s) * eps_s ** 2
    assert ustar == pytest.approx(0.4606553, abs=1e-7)
    assert g(ustar) == pytest.approx(2.0100189, abs=1e-7)
    us = np.linspace(0.01, 0.99, 197)
    assert max(g(u) for u in us) <= g(ustar) + 1e-12
    # value, first and second derivative of g at u=1 from both sides: 1, -2, 6
    h = 1e-4
    for side in (-1, +1):
        g0, g1, g2 = g(1.0), g(1 + side * h), g(1 + 2 * side * h)
        d1 = side * (-3 * g0 + 4 * g1 - g2) / (2 * h)
        d2 = (g0 - 2 * g1 + g2) / h ** 2
        assert g0 == pytest.approx(1.0, abs=1e-14)
        assert d1 == pytest.approx(-2.0, abs=2e-6)
        assert d2 == pytest.approx(6.0, abs=2e-2)


def test_p11_spline_matches_small_scale_plummer(oracle_mod):
    # "spline softening length is 2.16 eps_p to match the small-scale Plummer force"
    eps_p = 0.01
    r = 1e-10
    ratio = oracle_mod.force_factor(r, 2.16 * eps_p) / oracle_mod.plummer_factor(r, eps_p)
    assert ratio == pytest.approx(10 / 2.16 ** 3, rel=1e-6)
    assert abs(ratio - 1) < 0.01
    # far outside, both are Newtonian
    assert oracle_mod.force_factor(1.0, 2.16 * eps_p) == pytest.approx(1.0, rel=1e-15)


# ---------------------------------------------------------------- P2
def test_p2_cutoff_is_by_cell_not_distance(oracle_mod):
    cpd, R, eps_p = 16, 2, 1e-3
    c = 1.0 / cpd
    # cells 4 and 7 along x: delta = 3 = R+1 -> no interaction although distance ~ 2.0 cells
    x1 = [4 * c + 0.999 * c, 0.3, 0.3]
    x2 = [7 * c + 0.001 * c, 0.3, 0.3]
    _, acc, pairs = _two(oracle_mod, x1, x2, cpd, R, eps_p)
    assert pairs == 0 and np.all(acc == 0)
    # cells 4 and 6: delta = 2 = R -> Newtonian even at distance ~ 2.99 cells
    x1 = [4 * c + 0.001 * c, 0.3, 0.3]
    x2 = [6 * c + 0.999 * c, 0.3, 0.3]
    pos, acc, pairs = _two(oracle_mod, x1, x2, cpd, R, eps_p)
    r = pos[1, 0] - pos[0, 0]
    assert pairs == 2
    assert acc[0, 0] == pytest.approx(1 / r ** 2, rel=1e-12)
    assert acc[1, 0] == pytest.approx(-1 / r ** 2, rel=1e-12)
    assert np.all(acc[:, 1:] == 0)


# ---------------------------------------------------------------- P3
def test_p3_periodic_wrap(oracle_mod):
    cpd, R, eps_p = 7, 2, 1e-4
    pos, acc, pairs = _two(oracle_mod, [0.01, 0.5, 0.5], [0.99, 0.5, 0.5], cpd, R, eps_p)
    r = (pos[0, 0] + 1.0) - pos[1, 0]          # across the boundary
    assert pairs == 2
    assert acc[0, 0] == pytest.approx(-1 / r ** 2, rel=1e-9)   # particle 0 pulled to -x
    assert acc[1, 0] == pytest.approx(+1 / r ** 2, rel=1e-9)
    # all three axes at once, diagonal wrap
    pos, acc, _ = _two(oracle_mod, [0.01, 0.02, 0.98], [0.98, 0.99, 0.03], cpd, R, eps_p)
    d = (pos[1] - pos[0]) - np.round(pos[1] - pos[0])
    f = d / np.linalg.norm(d) ** 3
    assert np.allclose(acc[0], f, rtol=1e-9)


# ---------------------------------------------------------------- P4
@pytest.mark.parametrize("cpd,R", [(7, 2), (9, 3), (6, 2)])
def test_p4_one_particle_per_cell_lattice_is_force_free(oracle_mod, cpd, R):
    g = (np.arange(cpd) + 0.37) / cpd
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    acc, pairs = oracle_mod.accel(pos, cpd, R, 0.01 / cpd, gm=1.0)
    assert pairs == cpd ** 3 * ((2 * R + 1) ** 3 - 1)
    scale = cpd ** 2                          # one neighbour at one cell distance
    # float32 rounding of (i+0.37)/cpd (~3e-8) breaks the exact symmetry: |da| ~ 2 cpd^3 * 3e-8 * few
    assert np.abs(acc).max() <= 1e-5 * scale
    # exactly symmetric inputs (positions representable in float32): cpd = 8
    for Rx, o in ((2, 0.5), (3, 0.25), (2, 0.0)):
        g = (np.arange(8) + o) / 8
        pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
        acc, _ = oracle_mod.accel(pos, 8, Rx, 0.01, gm=1.0)
        assert np.abs(acc).max() <= 1e-13 * 64


def test_p4b_commensurate_lattice_identical_across_cells(oracle_mod):
    cpd, n = 8, 2                              # 2^3 particles per cell
    g = (np.arange(cpd * n) + 0.5) / (cpd * n)
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    acc, _ = oracle_mod.accel(pos, cpd, 2, 0.002, gm=1.0)
    A = acc.reshape(cpd, n, cpd, n, cpd, n, 3).transpose(0, 2, 4, 1, 3, 5, 6).reshape(cpd ** 3, n ** 3, 3)
    spread = np.abs(A - A[0]).max()
    assert spread <= 1e-12 * np.abs(A).max()
    assert np.abs(A[0].sum(0)).max() <= 1e-12 * np.abs(A).max()
    assert np.abs(A).max() > 1.0               # and it is NOT zero (stencil centred on the cell)


# ---------------------------------------------------------------- P5, P6, P7
def _brute_force(pos32, cpd, R, eps_p, gm):
    """All-pairs O(N^2), particle minimum image, masked to wrapped cell delta <= R per axis.
    Written independently of the oracle: float64 numpy, global coordinates."""
    x = pos32.astype(np.float64)
    N = len(x)
    ci = np.floor(x * cpd).astype(np.int64) % cpd
    eps_s = 2.16 * eps_p
    acc = np.zeros((N, 3))
    npairs = 0
    for i in range(N):
        d = x - x[i]
        d -= np.round(d)
        dc = np.abs(ci - ci[i])
        dc = np.minimum(dc, cpd - dc)
        m = np.all(dc <= R, axis=1)
        m[i] = False
        npairs += int(m.sum())
        dd = d[m]
        r = np.sqrt((dd ** 2).sum(1))
        u = r / eps_s
        with np.errstate(divide="ignore", invalid="ignore"):
            f = np.where(u < 1, (10 - 15 * u + 6 * u * u) / eps_s ** 3, 1 / r ** 3)
        f[r == 0] = 0
        acc[i] = gm * (f[:, None] * dd).sum(0)
    return acc, npairs


@pytest.mark.parametrize("cpd,R,N,seed", [(7, 2, 1500, 1), (6, 2, 900, 2), (9, 3, 1200, 3), (8, 3, 700, 4)])
def test_p6_brute_force_masked_all_pairs(oracle_mod, cpd, R, N, seed):
    assert cpd >= 2 * R + 2          # minimum image == cell-pair image only then (reading S3)
    pos = W.uniform(N, seed)
    eps_p = 0.05 / cpd
    acc, pairs = oracle_mod.accel(pos, cpd, R, eps_p)
    ref, npairs = _brute_force(pos, cpd, R, eps_p, 1.0 / N)
    rms = np.sqrt((ref ** 2).sum(1).mean())
    assert pairs == npairs
    assert np.abs(acc - ref).max() <= 1e-11 * rms


def test_p6_config1_in_full(oracle_mod):
    c = W.CONFIGS[1]
    pos = W.make_positions(c)
    acc, pairs = oracle_mod.accel(pos, c.cpd, c.R, c.eps_p)
    sel = np.random.default_rng(5).choice(c.N, 400, replace=False)
    x = pos.astype(np.float64)
    ci = np.floor(x * c.cpd).astype(np.int64) % c.cpd
    eps_s = 2.16 * c.eps_p
    for i in sel:
        d = x - x[i]; d -= np.round(d)
        dc = np.abs(ci - ci[i]); dc = np.minimum(dc, c.cpd - dc)
        m = np.all(dc <= c.R, axis=1); m[i] = False
        dd = d[m]; r = np.sqrt((dd ** 2).sum(1)); u = r / eps_s
        f = np.where(u < 1, (10 - 15 * u + 6 * u * u) / eps_s ** 3, 1 / np.maximum(r, 1e-300) ** 3)
        ref = c.gm * (f[:, None] * dd).sum(0)
        assert np.abs(acc[i] - ref).max() <= 1e-11 * np.abs(acc).max()
    assert pairs == 38_594_114       # BASELINE.md pair table, config 1, seed 0


def _box_filter_pairs(counts3, R):
    """P7: pairs = sum_c n_c (B*n)_c - N with B the periodic (2R+1)^3 box filter."""
    f = counts3.astype(np.int64)
    for ax in range(3):
        f = sum(np.roll(f, s, axis=ax) for s in range(-R, R + 1))
    return int((counts3.astype(np.int64) * f).sum() - counts3.sum())


@pytest.mark.parametrize("kind,cpd,R", [("uniform", 7, 2), ("uniform", 11, 3), ("plummer", 12, 2), ("uniform", 5, 2)])
def test_p5_p7_momentum_and_pair_count(oracle_mod, kind, cpd, R):
    N = 3000
    pos = W.uniform(N, 7) if kind == "uniform" else W.plummer_mixture(N, cpd, 7, n_spheres=5)
    acc, pairs = oracle_mod.accel(pos, cpd, R, 0.02 / cpd)
    cell, _ = oracle_mod.bin_particles(pos, cpd)
    counts = np.bincount(cell, minlength=cpd ** 3).reshape(cpd, cpd, cpd)
    offsets, _ = oracle_mod.cell_lists(cell, cpd)
    assert pairs == _box_filter_pairs(counts, R) == oracle_mod.pair_count(offsets, cpd, R)
    assert np.abs(acc.sum(0)).max() <= 1e-13 * np.abs(acc).sum()


# ---------------------------------------------------------------- P8
@pytest.mark.parametrize("cpd,R", [(5, 2), (7, 3), (3, 1)])
def test_p8_min_cpd_is_plain_all_pairs_with_cell_pair_image(oracle_mod, cpd, R):
    N = 600
    pos = W.uniform(N, 11)
    eps_p = 0.03 / cpd
    acc, pairs = oracle_mod.accel(pos, cpd, R, eps_p, gm=1.0)
    assert pairs == N * (N - 1)
    # plain direct sum; image = the cell-pair image: cell delta folded into [-R, R]
    x = pos.astype(np.float64)
    t = x * cpd
    ci = np.floor(t)
    off = (t - ci - 0.5) / cpd
    eps_s = 2.16 * eps_p
    ref = np.zeros_like(x)
    for i in range(N):
        dcell = ci - ci[i]
        dcell = (dcell + R) % cpd - R
        d = (off - off[i]) + dcell / cpd
        r = np.sqrt((d ** 2).sum(1)); r[i] = 1.0
        u = r / eps_s
        f = np.where(u < 1, (10 - 15 * u + 6 * u * u) / eps_s ** 3, 1 / r ** 3); f[i] = 0
        ref[i] = (f[:, None] * d).sum(0)
    assert np.abs(acc - ref).max() <= 1e-11 * np.sqrt((ref ** 2).sum(1).mean())


def test_p8_open_boundary_textbook_direct_sum(oracle_mod):
    # all particles inside the central cell of a big grid, eps tiny -> textbook Newtonian sum
    cpd, R, N = 9, 2, 200
    rng = np.random.default_rng(3)
    pos = ((4 + rng.random((N, 3))) / cpd).astype(np.float32)
    acc, _ = oracle_mod.accel(pos, cpd, R, 1e-7, gm=1.0)
    x = pos.astype(np.float64)
    d = x[None] - x[:, None]
    r2 = (d ** 2).sum(-1); np.fill_diagonal(r2, 1.0)
    f = r2 ** -1.5; np.fill_diagonal(f, 0.0)
    ref = (f[..., None] * d).sum(1)
    assert np.allclose(acc, ref, rtol=1e-9, atol=0)


# ---------------------------------------------------------------- P9, P10
def test_p9_translation_by_whole_cells(oracle_mod):
    cpd, R, N = 8, 2, 2500            # box = 1, cell = 1/8
    # positions on a 2^-20 grid: every whole-cell shift and wrap is then exact in float32
    pos = (np.floor(W.uniform(N, 21).astype(np.float64) * 2 ** 20) / 2 ** 20).astype(np.float32)
    acc0, _ = oracle_mod.accel(pos, cpd, R, 0.004)
    sh = np.array([3, 5, 6], dtype=np.float64) / cpd
    p2 = pos.astype(np.float64) + sh
    p2 -= np.floor(p2)
    assert np.array_equal(p2.astype(np.float32).astype(np.float64), p2)
    acc1, _ = oracle_mod.accel(p2.astype(np.float32), cpd, R, 0.004)
    assert np.abs(acc1 - acc0).max() <= 1e-13 * np.abs(acc0).max()


def test_p10_input_order_invariance(oracle_mod):
    c = W.scaled(W.CONFIGS[2], 7)
    pos = W.make_positions(c)
    acc0, _ = oracle_mod.accel(pos, c.cpd, c.R, c.eps_p)
    perm = np.random.default_rng(9).permutation(c.N)
    acc1, _ = oracle_mod.accel(pos[perm], c.cpd, c.R, c.eps_p)
    assert np.abs(acc1 - acc0[perm]).max() <= 1e-13 * np.abs(acc0).max()


# ---------------------------------------------------------------- binning, neighbour lists
def test_binning_half_open_cells_and_offsets(oracle_mod):
    cpd = 8
    pos = np.array([[0.0, 0.125, 0.2499999], [0.25, 0.9999999, 0.5], [1.0, -0.125, 1.125]], dtype=np.float32)
    cell, off = oracle_mod.bin_particles(pos, cpd)
    c3 = np.stack([cell // 64, (cell // 8) % 8, cell % 8], -1)
    assert c3.tolist() == [[0, 1, 1], [2, 7, 4], [0, 7, 1]]     # floor, half-open, periodic wrap
    assert np.all(off >= -0.5 / cpd) and np.all(off < 0.5 / cpd)
    assert off[0, 0] == -0.5 / cpd and off[1, 2] == -0.5 / cpd
    offsets, order = oracle_mod.cell_lists(np.array([3, 1, 3, 0, 1], dtype=np.int32), 2)
    assert offsets.tolist() == [0, 1, 3, 3, 5, 5, 5, 5, 5]
    assert order.tolist() == [3, 1, 4, 0, 2]                    # stable


def test_neighbor_lists(oracle_mod):
    cpd, R = 7, 2
    ids, img = oracle_mod.neighbors(cpd, R, (0 * 7 + 6) * 7 + 3)
    assert len(ids) == 125 and len(set(ids.tolist())) == 125
    # first entry: (a,b,c) = (-2,-2,-2) -> cell (5,4,1), image (-1,0,0)
    assert ids[0] == (5 * 7 + 4) * 7 + 1 and img[0].tolist() == [-1, 0, 0]
    # centre entry is the cell itself
    assert ids[62] == (0 * 7 + 6) * 7 + 3 and img[62].tolist() == [0, 0, 0]
    # last: (2,2,2) -> (2,1,5), image (0,1,0)
    assert ids[124] == (2 * 7 + 1) * 7 + 5 and img[124].tolist() == [0, 1, 0]
    # symmetry of the neighbour relation
    for c in (0, 100, 342):
        for n in oracle_mod.neighbors(cpd, R, c)[0]:
            assert c in oracle_mod.neighbors(cpd, R, int(n))[0]


def test_bad_arguments(oracle_mod):
    pos = W.uniform(10, 0)
    with pytest.raises(ValueError):
        oracle_mod.accel(pos, 4, 2, 0.01)              # cpd < 2R+1
    bad = pos.copy(); bad[3, 1] = np.nan
    with pytest.raises(ValueError):
        oracle_mod.accel(bad, 7, 2, 0.01)
    acc, pairs = oracle_mod.accel(np.zeros((0, 3), np.float32), 7, 2, 0.01)
    assert pairs == 0 and acc.shape == (0, 3)


def test_sink_cell_subset_matches_full(oracle_mod):
    c = W.scaled(W.CONFIGS[3], 9)
    pos = W.make_positions(c)
    full, _ = oracle_mod.accel(pos, c.cpd, c.R, c.eps_p)
    cells = np.array([0, 17, 400, 728], dtype=np.int32)
    sub, _ = oracle_mod.accel(pos, c.cpd, c.R, c.eps_p, sink_cells=cells)
    cell, _ = oracle_mod.bin_particles(pos, c.cpd)
    m = np.isin(cell, cells)
    assert m.any()
    assert np.array_equal(sub[m], full[m]) and np.all(sub[~m] == 0)
