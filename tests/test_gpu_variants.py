"""Parity of the kernel variants (C ABI: nf_set_softening, nf_set_density_radius, nf_accel4)
against ``oracle.accel_variant`` on the same seeded inputs: Plummer softening (Eq. 2), no softening
(PAPER.md:218), the FoF-scale density estimate.

Bars: accelerations as in tests/test_gpu_parity.py (north_star: per particle |da| <= 1e-5 rms|a|,
median relative error <= 2e-6).  Density estimate: a float32 sum of at most a few
hundred non-negative terms b^2 - r^2, each carrying the float32 rounding of r^2 (DESIGN.md
"Variants"): per particle |dw| <= 2e-5 * rms(w), median relative error <= 2e-6.
"""
import numpy as np
import pytest

from paper_2110_11392_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_ABS, TOL_MED = 1e-5, 2e-6
TOL_W_ABS, TOL_W_MED = 2e-5, 2e-6


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback exists)"
    torch.cuda.set_device(0)
    return torch


@pytest.fixture(scope="module")
def NF():
    from paper_2110_11392_b200.binding import NearField
    return NearField


def run(torch, NF, pos, cfg, law="spline", b=0.0, opts=None):
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        nf.set_softening(law)
        nf.set_density_radius(b)
        for k, v in (opts or {}).items():
            nf.set_option(k, v)
        d_pos = torch.from_numpy(pos).cuda()
        if b > 0:
            out = nf.accel4(d_pos)
            nf.sync()
            out = out.cpu().numpy().astype(np.float64)
            return out[:, :3], out[:, 3], nf.close_radius()
        acc = nf.accel(d_pos)
        nf.sync()
        return acc.cpu().numpy().astype(np.float64), None, nf.close_radius()


def check_acc(got, ref, label):
    d = np.linalg.norm(got - ref, axis=1)
    a = np.linalg.norm(ref, axis=1)
    rms = np.sqrt((a ** 2).mean())
    assert np.isfinite(got).all(), label
    worst = d.max() / rms
    med = np.median(d[a > 0] / a[a > 0])
    assert worst <= TOL_ABS, f"{label}: max |da| = {worst:.3e} rms|a|"
    assert med <= TOL_MED, f"{label}: median relative error {med:.3e}"


def check_dens(got, ref, label):
    assert np.isfinite(got).all(), label
    rms = np.sqrt((ref ** 2).mean())
    worst = np.abs(got - ref).max() / rms
    nz = ref > 1e-3 * rms
    med = np.median(np.abs(got - ref)[nz] / ref[nz])
    assert worst <= TOL_W_ABS, f"{label}: max |dw| = {worst:.3e} rms(w)"
    assert med <= TOL_W_MED, f"{label}: median relative density error {med:.3e}"
    assert np.all(got[ref == 0] <= TOL_W_ABS * rms)


CASES = [
    ("cfg1 full", W.CONFIGS[1]),
    ("cfg2 @cpd13", W.scaled(W.CONFIGS[2], 13)),
    ("cfg3 @cpd10", W.scaled(W.CONFIGS[3], 10)),
    ("cfg4 @cpd9", W.scaled(W.CONFIGS[4], 9)),
    ("cfg5 @cpd9 R3", W.scaled(W.CONFIGS[5], 9)),
]


@pytest.mark.parametrize("label,cfg", CASES, ids=[c[0] for c in CASES])
def test_plummer_softening(torch_cuda, NF, oracle_mod, label, cfg):
    pos = W.make_positions(cfg)
    got, _, rc = run(torch_cuda, NF, pos, cfg, law="plummer")
    ref, _, _ = oracle_mod.accel_variant(pos, cfg.cpd, cfg.R, cfg.eps_p, law="plummer")
    check_acc(got, ref, f"plummer {label} (rc={rc:.3g})")
    if rc == 0:                                    # also through the close-pair regime (self pairs told by d == 0)
        got2, _, rc2 = run(torch_cuda, NF, pos, cfg, law="plummer", opts={"rc_cells": 0.05})
        assert rc2 > 0
        check_acc(got2, ref, f"plummer {label} (forced rc={rc2:.3g})")
    # and it is not the spline: the two laws differ where particles are closer than a few eps
    spl, _ = oracle_mod.accel(pos, cfg.cpd, cfg.R, cfg.eps_p)
    assert np.abs(spl - ref).max() > 1e-4 * np.sqrt((ref ** 2).sum(1).mean())


@pytest.mark.parametrize("label,cfg", CASES, ids=[c[0] for c in CASES])
def test_unsoftened_newtonian_law(torch_cuda, NF, oracle_mod, label, cfg):
    """NF_SOFT_NEWTON ("Newtonian gravity, or a softened form thereof"): r/|r|^3 for every
    pair, the closest ones through the double-precision close-pair path; eps_p does not enter."""
    pos = W.make_positions(cfg)
    got, _, rc = run(torch_cuda, NF, pos, cfg, law="newton")
    ref, _, _ = oracle_mod.accel_variant(pos, cfg.cpd, cfg.R, cfg.eps_p, law="newton")
    assert rc > 0
    check_acc(got, ref, f"newton {label} (rc={rc:.3g})")
    got0, _, rc0 = run(torch_cuda, NF, pos, cfg, law="newton", opts={"rc_cells": 0.0})      # asked for none: kept at the floor
    assert 0 < rc0 <= 1.01e-4 and np.isfinite(got0).all()
    # the f64 entry point follows the same law
    with NF(cfg.cpd, cfg.R, cfg.eps_p * 7.0, 1.0) as nf:                                     # another eps: ignored
        nf.set_softening("newton")
        a64 = nf.accel_f64(torch_cuda.from_numpy(pos).cuda())
        nf.sync()
        a64 = a64.cpu().numpy()
    assert np.abs(a64 - ref).max() <= 1e-12 * np.sqrt((ref ** 2).sum(1).mean())


def test_newton_two_particles_and_coincident(torch_cuda, NF, oracle_mod):
    cfg = W.Config("n2", 8, 2, 0, "uniform", 0.01)
    for sep in (1e-5, 1e-3, 0.02, 0.11):
        for x1 in ((0.52, 0.58, 0.53), (0.4999, 0.56, 0.53)):                              # same cell / across a cell face
            pos = np.array([x1, np.array(x1) + sep * np.array([2.0, -1.0, 2.0]) / 3.0], dtype=np.float32)
            got, _, _ = run(torch_cuda, NF, pos, cfg, law="newton")
            ref, _, _ = oracle_mod.accel_variant(pos, cfg.cpd, cfg.R, cfg.eps_p, law="newton")
            assert np.allclose(got, ref, rtol=3e-6, atol=0), (sep, x1)
    pos = np.array([[0.3, 0.3, 0.3], [0.3, 0.3, 0.3], [0.35, 0.3, 0.3]], dtype=np.float32)     # a coincident pair: contributes 0
    got, _, _ = run(torch_cuda, NF, pos, cfg, law="newton")
    ref, _, _ = oracle_mod.accel_variant(pos, cfg.cpd, cfg.R, cfg.eps_p, law="newton")
    assert np.isfinite(got).all() and np.allclose(got, ref, rtol=3e-6)


@pytest.mark.parametrize("label,cfg", CASES, ids=[c[0] for c in CASES])
@pytest.mark.parametrize("bfrac", [0.35, 1.0], ids=["b=0.35cell", "b=1cell"])
def test_density_estimate(torch_cuda, NF, oracle_mod, label, cfg, bfrac):
    """b = 0.35 cell holds ~10-20 particles at 64 per cell (PAPER.md:503 'using 10-20 particles')."""
    pos = W.make_positions(cfg)
    b = bfrac * cfg.cell
    acc, dens, _ = run(torch_cuda, NF, pos, cfg, b=b)
    racc, rdens, _ = oracle_mod.accel_variant(pos, cfg.cpd, cfg.R, cfg.eps_p, density_b=b)
    check_acc(acc, racc, f"acc with density {label}")
    check_dens(dens, rdens, f"density {label} b={bfrac} cell")


def test_density_with_plummer_and_wide_radius(torch_cuda, NF, oracle_mod):
    """both variants at once; b > 1 cell widens the near-cell range (2 cells here)."""
    cfg = W.scaled(W.CONFIGS[2], 11)
    pos = W.make_positions(cfg)
    b = 1.6 * cfg.cell
    acc, dens, _ = run(torch_cuda, NF, pos, cfg, law="plummer", b=b)
    racc, rdens, _ = oracle_mod.accel_variant(pos, cfg.cpd, cfg.R, cfg.eps_p, law="plummer", density_b=b)
    check_acc(acc, racc, "plummer + density")
    check_dens(dens, rdens, "plummer + density")


def test_density_edge_cases(torch_cuda, NF, oracle_mod):
    cfg = W.Config("edge", 7, 2, 0, "uniform", 1e-3)
    b = 0.03
    # a lone particle, a coincident triple (each sees two at r = 0), a pair across the periodic boundary
    pos = np.array([[0.3, 0.3, 0.3], [0.6, 0.6, 0.6], [0.6, 0.6, 0.6], [0.6, 0.6, 0.6],
                    [0.005, 0.5, 0.5], [0.995, 0.5, 0.5]], dtype=np.float32)
    acc, dens, _ = run(torch_cuda, NF, pos, cfg, b=b)
    _, rdens, _ = oracle_mod.accel_variant(pos, cfg.cpd, cfg.R, cfg.eps_p, density_b=b)
    assert dens[0] == 0.0
    assert np.allclose(dens[1:4], 2 * b * b, rtol=1e-6)
    assert np.allclose(dens, rdens, rtol=1e-5, atol=1e-9)
    # radius 0: nf_accel4 leaves the 4th component alone and the accelerations are those of nf_accel
    a4, d4, _ = run(torch_cuda, NF, W.make_positions(W.CONFIGS[1]), W.CONFIGS[1], b=0.0)
    assert d4 is None


def test_variant_setters_reject_bad_arguments(torch_cuda, NF):
    from paper_2110_11392_b200.binding import NearFieldError, _L
    with NF(7, 2, 1e-3, 1.0) as nf:
        with pytest.raises(NearFieldError):
            nf._check(_L.nf_set_softening(nf._h, 7))
        with pytest.raises(NearFieldError):
            nf.set_density_radius(-1.0)
        with pytest.raises(NearFieldError):
            nf.set_density_radius(float("nan"))
