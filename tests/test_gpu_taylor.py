"""nf_taylor_accel (reading F1) against ``oracle.taylor_accel``: the kernel
evaluates in double (Horner in z, power tables in x and y) and rounds to float32 once, so the bar is
the float32 rounding of the result: per particle |da| <= 3e-7 * rms|a| (coefficients scaled so that
every order contributes)."""
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


def _coeffs(oracle_mod, cpd, order, seed):
    rng = np.random.default_rng(seed)
    idx = oracle_mod.multipole_index(order)
    return rng.normal(size=(cpd ** 3, len(idx))) * np.array([float(cpd) ** (a + b + c) for a, b, c in idx]), idx


CASES = [("cfg1 p8", W.CONFIGS[1], 8), ("cfg3 @cpd10 p8", W.scaled(W.CONFIGS[3], 10), 8), ("cfg4 @cpd9 p8", W.scaled(W.CONFIGS[4], 9), 8),
         ("cfg2 @cpd6 p3", W.scaled(W.CONFIGS[2], 6), 3), ("cfg2 @cpd6 p16", W.scaled(W.CONFIGS[2], 6), 16), ("cfg2 @cpd6 p0", W.scaled(W.CONFIGS[2], 6), 0)]


@pytest.mark.parametrize("label,cfg,order", CASES, ids=[c[0] for c in CASES])
def test_taylor_accel_matches_the_oracle(torch_cuda, NF, oracle_mod, label, cfg, order):
    pos = W.make_positions(cfg)
    T, idx = _coeffs(oracle_mod, cfg.cpd, order, 1)
    ref = oracle_mod.taylor_accel(pos, T, cfg.cpd, order)
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        d_pos = torch_cuda.from_numpy(pos).cuda()
        d_T = torch_cuda.from_numpy(T).cuda()
        acc = nf.taylor_accel(d_pos, d_T, order)
        near = nf.accel(d_pos)
        both = nf.taylor_accel(d_pos, d_T, order, acc=near.clone(), accumulate=True)
        nf.sync()
        got, near, both = acc.cpu().numpy(), near.cpu().numpy(), both.cpu().numpy()
    rms = np.sqrt((ref ** 2).sum(1).mean()) if order > 0 else 1.0
    assert np.isfinite(got).all()
    assert np.abs(got - ref).max() <= 3e-7 * rms, label          # float32 rounding of a result of size ~rms
    assert np.allclose(both, near + got, rtol=0, atol=2e-7 * (np.abs(near).max() + np.abs(got).max() + 1e-30))
    if order == 0:
        assert np.all(got == 0)


def test_taylor_uniform_field_and_empty(torch_cuda, NF, oracle_mod):
    cfg = W.CONFIGS[1]
    pos = W.make_positions(cfg)
    idx = oracle_mod.multipole_index(8)
    T = np.zeros((cfg.cpd ** 3, len(idx)))
    T[:, idx.index((0, 1, 0))] = 0.25
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        acc = nf.taylor_accel(torch_cuda.from_numpy(pos).cuda(), torch_cuda.from_numpy(T).cuda(), 8)
        e = torch_cuda.zeros((0, 3), dtype=torch_cuda.float32, device="cuda")
        nf.taylor_accel(e, torch_cuda.from_numpy(T).cuda(), 8)
        nf.sync()
    assert np.array_equal(acc.cpu().numpy(), np.tile(np.float32([0, -0.25, 0]), (cfg.N, 1)))
