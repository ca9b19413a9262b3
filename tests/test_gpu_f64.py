"""nf_accel_f64 (the double-precision direct sum on the GPU) against the CPU oracle, and the
float32 product path against it on EVERY particle of full-size inputs -- the whole-input check the
CPU oracle cannot reach (it covers samples of configs 3-5 in tests/test_gpu_parity.py)."""
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


SMALL = [("cfg1 full", W.CONFIGS[1]), ("cfg3 @cpd10", W.scaled(W.CONFIGS[3], 10)), ("cfg5 @cpd9 R3", W.scaled(W.CONFIGS[5], 9)),
         ("cfg2 @cpd5 (=2R+1)", W.scaled(W.CONFIGS[2], 5))]


@pytest.mark.parametrize("label,cfg", SMALL, ids=[s[0] for s in SMALL])
@pytest.mark.parametrize("law", ["spline", "plummer"])
def test_f64_path_equals_the_oracle(torch_cuda, NF, oracle_mod, label, cfg, law):
    """same definition, same precision: only the rounding order of a double sum differs."""
    pos = W.make_positions(cfg)
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        nf.set_softening(law)
        got = nf.accel_f64(torch_cuda.from_numpy(pos).cuda())
        nf.sync()
        got = got.cpu().numpy()
    ref, _, _ = oracle_mod.accel_variant(pos, cfg.cpd, cfg.R, cfg.eps_p, law=law)
    rms = np.sqrt((ref ** 2).sum(1).mean())
    assert np.abs(got - ref).max() <= 1e-12 * rms, label


def _f32_vs_f64(torch, NF, cfg, label):
    pos = torch.from_numpy(W.make_positions(cfg)).cuda()
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        a32 = nf.accel(pos)
        nf.sync()
        a64 = nf.accel_f64(pos)
        nf.sync()
    d = (a32.double() - a64).norm(dim=1)
    a = a64.norm(dim=1)
    rms = float((a * a).mean().sqrt())
    worst = float(d.max()) / rms
    med = float((d[a > 0] / a[a > 0]).median())
    assert bool(torch.isfinite(a32).all())
    assert worst <= 1e-5, f"{label}: max |da| = {worst:.3e} rms|a| over all {cfg.N} particles"
    assert med <= 2e-6, f"{label}: median relative error {med:.3e}"
    return worst, med


@pytest.mark.parametrize("k", [2, 3, 4, 5])
def test_full_size_configs_every_particle(torch_cuda, NF, k):
    """BASELINE.json configs 2-5 at FULL size (config 4: all 157 464 000 particles), in the launch
    configuration bench.py times: the north_star bar on every particle, against the GPU's own
    double-precision sum (which the test above ties to the oracle)."""
    cfg = W.CONFIGS[k]
    worst, med = _f32_vs_f64(torch_cuda, NF, cfg, f"config {k} (N={cfg.N})")
    print(f"config {k}: max |da| = {worst:.3e} rms|a|, median rel = {med:.3e}")
    torch_cuda.cuda.empty_cache()
