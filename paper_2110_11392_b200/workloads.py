"""Seeded synthetic input generators for the Abacus near-field workloads.

This module is the ONLY code shared between the CPU oracle (``oracle/``) and the CUDA
path (``paper_2110_11392_b200/csrc``).  It holds none of the method's arithmetic: no
binning, no force law, no neighbour logic -- only recipes that turn a seed into a
float32 ``pos[N][3]`` array in ``[0, box)`` plus the scalar parameters of a config.

The five configs are ``BASELINE.json:configs`` (recipes: DESIGN.md "Input recipe",
following SURVEY.md section 8(d)).  They stand in for the paper's own workloads
(AbacusSummit states, the 512^3 LCDM snapshot of PAPER.md:318), which are not
available: the shapes are the paper's -- 30-100 particles per cell,
R = 2, softening = spacing/40, clustered late-time
states.

Generator: numpy ``default_rng(seed)`` (PCG64).  Positions are produced in float64,
wrapped into [0, 1), cast to float32, and any value that rounds up to 1.0 is set to 0.0.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

BOX = 1.0


@dataclass(frozen=True)
class Config:
    """Scalar parameters of one workload (``BASELINE.json:configs[k-1]``)."""

    name: str
    cpd: int          # cells per dimension, K in PAPER.md:72
    R: int            # near-field radius in cells
    N: int            # particle count
    kind: str         # "uniform" | "lattice" | "plummer"
    eps_p: float      # Plummer-equivalent softening length, box units
    box: float = BOX
    seed: int = 0
    n_spheres: int = 20_000   # "plummer" kind only

    @property
    def gm(self) -> float:
        """G*m with G = 1 and equal masses 1/N (BASELINE.json config 1)."""
        return 1.0 / self.N

    @property
    def cell(self) -> float:
        return self.box / self.cpd


def _spacing_eps(N: int) -> float:
    # eps_p = (mean interparticle spacing)/40
    return (BOX / N ** (1.0 / 3.0)) / 40.0


CONFIGS = {
    1: Config("cfg1_cpd7_uniform", 7, 2, 10_290, "uniform", 0.1 * BOX / 7),
    2: Config("cfg2_cpd35_uniform", 35, 2, 1_715_000, "uniform", _spacing_eps(1_715_000)),
    3: Config("cfg3_cpd63_plummer", 63, 2, 64 * 63 ** 3, "plummer", _spacing_eps(64 * 63 ** 3)),
    4: Config("cfg4_cpd135_zeldovich", 135, 2, 540 ** 3, "lattice", _spacing_eps(540 ** 3)),
    5: Config("cfg5_cpd45_R3_plummer", 45, 3, 128 * 45 ** 3, "plummer", _spacing_eps(128 * 45 ** 3)),
}


def _finish(p64: np.ndarray) -> np.ndarray:
    """wrap to [0,1) in float64, cast to float32, fold values that round to 1.0 back to 0.0."""
    p64 -= np.floor(p64)
    p32 = p64.astype(np.float32)
    p32[p32 >= 1.0] = 0.0
    return p32


def uniform(N: int, seed: int = 0) -> np.ndarray:
    """iid uniform positions: ``default_rng(seed).random((N, 3))`` (configs 1, 2)."""
    return _finish(np.random.default_rng(seed).random((N, 3)))


def displaced_lattice(n_side: int, sigma: float, seed: int = 0, chunk_planes: int = 8) -> np.ndarray:
    """Cubic lattice ``(i + 1/2)/n_side`` (x slowest, z fastest) plus iid Gaussian
    displacements of standard deviation ``sigma`` (box units) per component (config 4:
    a synthetic stand-in for a Zel'dovich-displaced lattice).  Generated in x-plane chunks
    from ONE rng stream, so the result does not depend on ``chunk_planes``."""
    rng = np.random.default_rng(seed)
    N = n_side ** 3
    out = np.empty((N, 3), dtype=np.float32)
    g = (np.arange(n_side, dtype=np.float64) + 0.5) / n_side
    plane = n_side * n_side
    yz = np.empty((plane, 2), dtype=np.float64)
    yz[:, 0] = np.repeat(g, n_side)
    yz[:, 1] = np.tile(g, n_side)
    for i0 in range(0, n_side, chunk_planes):
        i1 = min(n_side, i0 + chunk_planes)
        m = (i1 - i0) * plane
        p = rng.standard_normal((m, 3))
        p *= sigma
        p[:, 0] += np.repeat(g[i0:i1], plane)
        p[:, 1] += np.tile(yz[:, 0], i1 - i0)
        p[:, 2] += np.tile(yz[:, 1], i1 - i0)
        out[i0 * plane:i1 * plane] = _finish(p)
    return out


def plummer_mixture(N: int, cpd: int, seed: int = 0, n_spheres: int = 20_000,
                    frac_clustered: float = 0.7) -> np.ndarray:
    """Clustered mixture of configs 3 and 5: ``frac_clustered`` of the particles in
    ``n_spheres`` Plummer spheres with random centres, sphere masses M in [1, 1000] drawn
    from dN/dM ~ M^-1.9, scale radius a = 0.05 cell * M^(1/3) (0.05 .. 0.5 cell), particle
    count per sphere proportional to M (largest-remainder rounding), radii from the inverse
    of M(<r)/M = r^3/(r^2+a^2)^(3/2) truncated at 10 a, isotropic directions; the rest
    uniform.  Sphere particles come first in the output, then the background."""
    rng = np.random.default_rng(seed)
    cell = BOX / cpd
    n_cl = int(round(frac_clustered * N))
    u = rng.random(n_spheres)
    M = (1.0 + u * (1000.0 ** -0.9 - 1.0)) ** (-1.0 / 0.9)
    a = 0.05 * cell * M ** (1.0 / 3.0)
    share = M / M.sum() * n_cl
    cnt = np.floor(share).astype(np.int64)
    rem = n_cl - int(cnt.sum())
    if rem > 0:
        order = np.argsort(-(share - cnt), kind="stable")
        cnt[order[:rem]] += 1
    centres = rng.random((n_spheres, 3))
    out = np.empty((N, 3), dtype=np.float32)
    sph = np.repeat(np.arange(n_spheres), cnt)
    step = 4_000_000
    xmax = 1000.0 / 101.0 ** 1.5          # mass fraction inside r = 10 a
    for s0 in range(0, n_cl, step):
        s1 = min(n_cl, s0 + step)
        idx = sph[s0:s1]
        X = rng.random(s1 - s0) * xmax
        X = np.maximum(X, 1e-300)
        r = a[idx] / np.sqrt(X ** (-2.0 / 3.0) - 1.0)
        mu = 2.0 * rng.random(s1 - s0) - 1.0
        phi = 2.0 * np.pi * rng.random(s1 - s0)
        st = np.sqrt(np.maximum(0.0, 1.0 - mu * mu))
        p = centres[idx].copy()
        p[:, 0] += r * st * np.cos(phi)
        p[:, 1] += r * st * np.sin(phi)
        p[:, 2] += r * mu
        out[s0:s1] = _finish(p)
    for s0 in range(n_cl, N, step):
        s1 = min(N, s0 + step)
        out[s0:s1] = _finish(rng.random((s1 - s0, 3)))
    return out


def make_positions(cfg: Config) -> np.ndarray:
    """float32 ``pos[N][3]`` in [0, 1) for one of ``CONFIGS``."""
    if cfg.kind == "uniform":
        return uniform(cfg.N, cfg.seed)
    if cfg.kind == "lattice":
        n_side = round(cfg.N ** (1.0 / 3.0))
        assert n_side ** 3 == cfg.N
        return displaced_lattice(n_side, 0.3 * cfg.cell, cfg.seed)
    if cfg.kind == "plummer":
        return plummer_mixture(cfg.N, cfg.cpd, cfg.seed, cfg.n_spheres)
    raise ValueError(cfg.kind)


def scaled(cfg: Config, cpd: int, seed: int | None = None) -> Config:
    """Same recipe and particles-per-cell as ``cfg`` on a smaller grid (parity-test
    sizes the oracle finishes in seconds).  Lattice configs keep 4 particles per cell per
    axis; the others keep N/cpd^3.  eps_p follows the spacing/40 rule (config 1 keeps
    0.1 cell); the number of Plummer spheres scales with the volume in cells."""
    ppc = cfg.N // cfg.cpd ** 3
    N = ppc * cpd ** 3
    eps = 0.1 * BOX / cpd if cfg is CONFIGS[1] else _spacing_eps(N)
    nsph = max(1, round(cfg.n_spheres * (cpd / cfg.cpd) ** 3))
    return Config(f"{cfg.name}@cpd{cpd}", cpd, cfg.R, N, cfg.kind, eps, cfg.box,
                  cfg.seed if seed is None else seed, nsph)
