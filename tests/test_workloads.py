"""Seeded input generators: determinism, ranges, the recipes' stated properties."""
import numpy as np
import pytest

from paper_2110_11392_b200 import workloads as W


def _box_filter_pairs(counts3, R):
    f = counts3.astype(np.int64)
    for ax in range(3):
        f = sum(np.roll(f, s, axis=ax) for s in range(-R, R + 1))
    return int((counts3.astype(np.int64) * f).sum() - counts3.sum())


def _counts(pos, cpd):
    c = np.floor(pos.astype(np.float64) * cpd).astype(np.int64) % cpd
    key = (c[:, 0] * cpd + c[:, 1]) * cpd + c[:, 2]
    return np.bincount(key, minlength=cpd ** 3).reshape(cpd, cpd, cpd)


def test_config_table_matches_baseline_json():
    c = W.CONFIGS
    assert (c[1].cpd, c[1].R, c[1].N) == (7, 2, 10_290)
    assert (c[2].cpd, c[2].R, c[2].N) == (35, 2, 1_715_000)
    assert (c[3].cpd, c[3].R, c[3].N) == (63, 2, 16_003_008)
    assert (c[4].cpd, c[4].R, c[4].N) == (135, 2, 157_464_000)
    assert (c[5].cpd, c[5].R, c[5].N) == (45, 3, 11_664_000)
    assert c[1].eps_p == pytest.approx(0.1 / 7)
    assert c[4].eps_p == pytest.approx(1 / 21600)
    assert c[2].eps_p == pytest.approx(1 / (40 * 1_715_000 ** (1 / 3)))
    assert c[4].gm == 1 / 157_464_000


@pytest.mark.parametrize("k", [1, 2])
def test_uniform_configs_pair_counts(k):
    cfg = W.CONFIGS[k]
    pos = W.make_positions(cfg)
    assert pos.dtype == np.float32 and pos.shape == (cfg.N, 3)
    assert pos.min() >= 0 and pos.max() < 1
    assert np.array_equal(pos, W.make_positions(cfg))
    expected = {1: 38_594_114, 2: 8_574_874_650}[k]          # BASELINE.md pair table, seed 0
    assert _box_filter_pairs(_counts(pos, cfg.cpd), cfg.R) == expected


def test_lattice_chunk_independent_and_occupancy():
    a = W.displaced_lattice(24, 0.3 / 6, seed=3, chunk_planes=5)
    b = W.displaced_lattice(24, 0.3 / 6, seed=3, chunk_planes=24)
    assert np.array_equal(a, b) and a.min() >= 0 and a.max() < 1
    cfg = W.scaled(W.CONFIGS[4], 9)
    pos = W.make_positions(cfg)
    cnt = _counts(pos, cfg.cpd)
    assert cfg.N == 64 * 9 ** 3 and cnt.sum() == cfg.N
    assert 30 < cnt.min() and cnt.max() < 110 and abs(np.median(cnt) - 64) <= 3      # 34..105, median 64
    # zero displacement reproduces the lattice exactly: 4 per cell per axis
    lat = W.displaced_lattice(16, 0.0)
    assert np.all(_counts(lat, 4) == 64)


def test_plummer_mixture_is_clustered_and_deterministic():
    cfg = W.scaled(W.CONFIGS[3], 12)
    pos = W.make_positions(cfg)
    assert np.array_equal(pos, W.make_positions(cfg))
    assert pos.shape == (64 * 12 ** 3, 3) and pos.min() >= 0 and pos.max() < 1
    cnt = _counts(pos, cfg.cpd)
    assert cnt.max() > 10 * cnt.mean()                 # heavy cells (load-imbalance case)
    assert np.median(cnt) < cnt.mean()                 # skewed
    uniform_pairs = cfg.N * (cfg.N / cfg.cpd ** 3) * 125
    assert _box_filter_pairs(cnt, 2) > 1.3 * uniform_pairs
    other = W.make_positions(W.scaled(W.CONFIGS[3], 12, seed=1))
    assert not np.array_equal(pos, other)


def test_values_rounding_to_one_are_folded():
    p = W._finish(np.array([[0.99999999999, 1.0 - 1e-12, -1e-12]]))
    assert p.max() < 1.0 and p.min() >= 0.0
