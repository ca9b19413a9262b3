"""nf_multipoles (Eq. 4) against ``oracle.multipoles`` on the same seeded inputs.

Every element is a double sum of monomials in the same particle order on both sides; the kernel
forms x^a y^b z^c as (x^a y^b) z^c with the last product fused into the add (the FMA form of
PAPER.md:199), the oracle by the pseudo-code's running products, so terms differ by a few ulp
and sums by the rounding of n additions.  Bar per element, with S = sum_q |x^a y^b z^c| and n the cell's
occupancy: |dM| <= (1e-13 + 2.3e-16 n) S -- the second term is the forward error bound (n - 1) u S of a
recursive double sum (u = 2^-53), which a long cell needs for the ORACLE's sake: in the 8404-particle cell of the
clustered case (cfg3 @cpd10) the oracle's sequential sum is up to 1.3e-13 S from the exactly rounded sum (maximum
over the 165 columns, measured on the CPU against math.fsum; its bound there is (n - 1) u = 9.3e-13 S), i.e.
already past a flat 1e-13 S.  (Round 2 quoted "2.7e-11" here without a unit; no unit makes that figure right.)
The kernel adds 512-particle chunks and then the partials, so the dense cells are ALSO held against math.fsum of
the same double offsets, at 1e-13 S without the n term, on ALL columns (counts, a = b = c = 0, are exact)."""
import numpy as np
import pytest

from paper_2110_11392_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    return torch


@pytest.fixture(scope="module")
def NF():
    from paper_2110_11392_b200.binding import NearField
    return NearField


def _abs_moments(pos, cpd, order, idx):
    t = pos.astype(np.float64) * cpd
    off = np.abs((t - np.floor(t) - 0.5) / cpd)
    c = np.floor(t).astype(np.int64) % cpd
    key = (c[:, 0] * cpd + c[:, 1]) * cpd + c[:, 2]
    out = np.empty((cpd ** 3, len(idx)))
    for col, (a, b, k) in enumerate(idx):
        out[:, col] = np.bincount(key, weights=off[:, 0] ** a * off[:, 1] ** b * off[:, 2] ** k, minlength=cpd ** 3)
    return out


CASES = [("cfg1 full p8", W.CONFIGS[1], 8), ("cfg2 @cpd13 p8", W.scaled(W.CONFIGS[2], 13), 8),
         ("cfg3 @cpd10 p8", W.scaled(W.CONFIGS[3], 10), 8), ("cfg4 @cpd9 p8", W.scaled(W.CONFIGS[4], 9), 8),
         ("cfg5 @cpd9 p4", W.scaled(W.CONFIGS[5], 9), 4), ("cfg2 @cpd6 p10", W.scaled(W.CONFIGS[2], 6), 10), ("cfg2 @cpd6 p16", W.scaled(W.CONFIGS[2], 6), 16),
         ("cfg2 @cpd6 p0", W.scaled(W.CONFIGS[2], 6), 0)]


@pytest.mark.parametrize("label,cfg,order", CASES, ids=[c[0] for c in CASES])
def test_multipoles_match_the_oracle(torch_cuda, NF, oracle_mod, label, cfg, order):
    pos = W.make_positions(cfg)
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        M = nf.multipoles(torch_cuda.from_numpy(pos).cuda(), order)
        nf.sync()
        got = M.cpu().numpy()
    ref = oracle_mod.multipoles(pos, cfg.cpd, order)
    idx = oracle_mod.multipole_index(order)
    assert got.shape == ref.shape == (cfg.cpd ** 3, len(idx))
    assert np.array_equal(got[:, 0], ref[:, 0])                              # occupancy: exact
    scale = _abs_moments(pos, cfg.cpd, order, idx)
    n = ref[:, :1]
    assert np.all(np.abs(got - ref) <= (1e-13 + 2.3e-16 * n) * scale + 1e-300), label
    # the cells of more than 512 particles (chunked on the GPU) against the exactly rounded sums
    import math
    t = pos.astype(np.float64) * cfg.cpd
    c = np.floor(t).astype(np.int64) % cfg.cpd
    key = (c[:, 0] * cfg.cpd + c[:, 1]) * cfg.cpd + c[:, 2]
    off = (t - np.floor(t) - 0.5) / cfg.cpd
    dense = np.flatnonzero(ref[:, 0] > 512)
    dense = dense[np.argsort(-ref[dense, 0], kind="stable")][:6]             # the six densest
    worst_k = worst_o = 0.0
    for cell in dense:
        o = off[key == cell]
        for col in range(len(idx)):                                          # every column of the basis
            a, b, k = idx[col]
            exact = math.fsum((o[:, 0] ** a * o[:, 1] ** b * o[:, 2] ** k).tolist())
            assert abs(got[cell, col] - exact) <= 1e-13 * scale[cell, col] + 1e-300, (label, int(cell), (a, b, k))
            if scale[cell, col] > 0:
                worst_k = max(worst_k, abs(got[cell, col] - exact) / scale[cell, col])
                worst_o = max(worst_o, abs(ref[cell, col] - exact) / scale[cell, col])
    if len(dense):
        print(f"MULTIPOLES {label}: {len(dense)} dense cells (n up to {int(ref[dense, 0].max())}), all {len(idx)} columns against math.fsum: "
              f"kernel {worst_k:.2e} S, oracle {worst_o:.2e} S")


def test_multipoles_edge_cases(torch_cuda, NF, oracle_mod):
    # empty input, a single particle, everything in one cell (all other cells must be zero-filled)
    with NF(7, 2, 1e-3, 1.0) as nf:
        M0 = nf.multipoles(torch_cuda.zeros((0, 3), dtype=torch_cuda.float32, device="cuda"), 8)
        nf.sync()
        assert M0.shape == (343, 165) and float(M0.abs().sum()) == 0.0
        rng = np.random.default_rng(3)
        pos = (0.5 + (rng.random((777, 3)) - 0.5) / 7.5).astype(np.float32)     # inside the central cell
        M = nf.multipoles(torch_cuda.from_numpy(pos).cuda(), 8)
        nf.sync()
        got = M.cpu().numpy()
    ref = oracle_mod.multipoles(pos, 7, 8)
    key = (3 * 7 + 3) * 7 + 3
    assert got[key, 0] == 777 and np.count_nonzero(np.delete(got, key, axis=0)) == 0
    assert np.allclose(got, ref, rtol=1e-12, atol=1e-30)


def test_multipoles_chunk_boundaries(torch_cuda, NF, oracle_mod):
    """cells on either side of the lane limit (1024) and of the 512-particle chunk size, shuffled input"""
    import math
    rng = np.random.default_rng(12)
    cpd = 5
    sizes = {(0, 0, 0): 1024, (1, 1, 1): 1025, (2, 2, 2): 1536, (3, 3, 3): 2049, (4, 4, 4): 511, (0, 4, 2): 513, (2, 0, 3): 5000}
    pos = np.concatenate([((np.array(c) + rng.random((n, 3))) / cpd) for c, n in sizes.items()])
    pos = pos[rng.permutation(len(pos))].astype(np.float32)
    pos[pos >= 1.0] = 0.0
    with NF(cpd, 2, 1e-3, 1.0) as nf:
        M = nf.multipoles(torch_cuda.from_numpy(pos).cuda(), 8)
        nf.sync()
        got = M.cpu().numpy()
    ref = oracle_mod.multipoles(pos, cpd, 8)
    idx = oracle_mod.multipole_index(8)
    scale = _abs_moments(pos, cpd, 8, idx)
    assert np.array_equal(got[:, 0], ref[:, 0])
    assert np.all(np.abs(got - ref) <= (1e-13 + 2.3e-16 * ref[:, :1]) * scale + 1e-300)
    t = pos.astype(np.float64) * cpd
    c = np.floor(t).astype(np.int64) % cpd
    key = (c[:, 0] * cpd + c[:, 1]) * cpd + c[:, 2]
    off = (t - np.floor(t) - 0.5) / cpd
    for cell in np.flatnonzero(ref[:, 0] > 0):
        o = off[key == cell]
        for col in range(len(idx)):
            a, b, k = idx[col]
            exact = math.fsum((o[:, 0] ** a * o[:, 1] ** b * o[:, 2] ** k).tolist())
            assert abs(got[cell, col] - exact) <= 1e-13 * scale[cell, col] + 1e-300, (int(cell), (a, b, k))


def test_multipoles_full_size_config4_properties(torch_cuda, NF):
    """config 4 at full size (157 464 000 particles, 2 460 375 cells x 165 = 3.2 GB): properties that
    hold at any size -- M^{000} = occupancy (sums to N), |M^{abc}| <= n (cell/2)^(a+b+c), and the
    second moments x^2 + y^2 + z^2 summed over the box = N * <r^2> ~ N cell^2 / 4 for uniform offsets."""
    cfg = W.CONFIGS[4]
    pos = torch_cuda.from_numpy(W.make_positions(cfg)).cuda()
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        M = nf.multipoles(pos, 8)
        nf.sync()
    assert int(M[:, 0].sum().item()) == cfg.N
    idx = [(a, b, c) for a in range(9) for b in range(9 - a) for c in range(9 - a - b)]
    half = 0.5 * cfg.cell
    n = M[:, 0]
    for col in (idx.index((1, 0, 0)), idx.index((0, 2, 0)), idx.index((2, 2, 2)), idx.index((0, 0, 8)), idx.index((8, 0, 0))):
        a, b, c = idx[col]
        assert bool((M[:, col].abs() <= n * half ** (a + b + c) * (1 + 1e-12)).all())
    r2 = float((M[:, idx.index((2, 0, 0))] + M[:, idx.index((0, 2, 0))] + M[:, idx.index((0, 0, 2))]).sum().item())
    assert abs(r2 / (cfg.N * cfg.cell ** 2 / 4.0) - 1.0) < 0.01
