"""Ordering evidence for the interaction kernel's consumer-refilled copy ring ("Who may write
what, and when"; the paper's own guard against silent corruption is guard bytes; the kernel it protects
is PAPER.md:236).

compute-sanitizer's racecheck is not available on this pool, so the argument in DESIGN.md is backed by stress builds:
the same sources compiled with a ring of 2 stages refilled only by starved warps (-DNF_NSTAGE=2 -DNF_REFILL_BELOW=1:
every stage boundary is a hand-over under the lock, slots are reused at once) and with another residency and depth
(-DNF_MIN_CTAS=1 -DNF_NSTAGE=3: other register allocation, other interleaving of the warps).  The summation order of a
sink is fixed by the stage sequence of its block (stages are cut by NF_TILE, not by the ring depth) and each block is
processed by one CTA, so a race-free kernel gives the SAME BITS under every such build and on every repeat.  The test
compares, bit for bit, 20 repeats of the default build and 20 repeats of each stress build on the small parity cases
and on config 3 (clustered: the uneven warps that make the lock busy) at full size.

Each stress library is built into a copy of the package under tmp_path and run in a subprocess (as
tests/test_gpu_debug_bounds.py does); results come back as .npy files.
"""
import os
import shutil
import subprocess
import sys

import numpy as np
import pytest

from paper_2110_11392_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
REPEATS = 20

RUNNER = r'''
import sys, numpy as np, torch
import paper_2110_11392_b200.binding as B
from paper_2110_11392_b200 import workloads as W
out_dir, copy, repeats = sys.argv[1], sys.argv[2], int(sys.argv[3])
assert copy == "-" or B.lib_path().startswith(copy), B.lib_path()
CASES = [("cfg1", W.CONFIGS[1], {}), ("cfg2at13", W.scaled(W.CONFIGS[2], 13), {}), ("cfg3at10", W.scaled(W.CONFIGS[3], 10), {}),
         ("cfg5at9", W.scaled(W.CONFIGS[5], 9), {}), ("tiny_blocks", W.Config("s", 16, 2, 2 * 16 ** 3, "uniform", 1.0 / (2 * 16 ** 3) ** (1 / 3) / 40, seed=9), {}),
         ("cfg3at10_rc02", W.scaled(W.CONFIGS[3], 10), {"rc_cells": 0.2}), ("cfg3_full", W.CONFIGS[3], {})]
for label, cfg, opts in CASES:
    d = torch.from_numpy(W.make_positions(cfg)).cuda()
    with B.NearField(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        for k, v in opts.items():
            nf.set_option(k, v)
        first = nf.accel(d).clone(); nf.sync()
        for r in range(repeats - 1):
            again = nf.accel(d); nf.sync()
            assert torch.equal(again, first), (label, "repeat", r + 1)
        pairs = nf.interaction_count()
        deliv, self_meet = nf.delivered_pairs()
        assert self_meet == cfg.N and deliv - self_meet == pairs, label
    np.save(f"{out_dir}/{label}.npy", first.cpu().numpy())
print("RING-OK")
'''

VARIANTS = [("nstage2_refill1", ("-DNF_NSTAGE=2", "-DNF_REFILL_BELOW=1")), ("minctas1_nstage3", ("-DNF_MIN_CTAS=1", "-DNF_NSTAGE=3"))]


def _run(script_args, env, cwd):
    r = subprocess.run([sys.executable, "-c", RUNNER, *script_args], cwd=cwd, env=env, capture_output=True, text=True, timeout=1200)
    assert r.returncode == 0 and "RING-OK" in r.stdout, r.stdout[-2000:] + r.stderr[-4000:]


@pytest.mark.gpu
def test_stress_builds_of_the_copy_ring_give_the_default_builds_bits(tmp_path):
    from paper_2110_11392_b200 import build
    pkg_src = os.path.dirname(os.path.abspath(build.__file__))
    ref_dir = tmp_path / "default"
    ref_dir.mkdir()
    _run([str(ref_dir), "-", str(REPEATS)], dict(os.environ, PYTHONPATH=ROOT), ROOT)          # the in-tree default build
    names = sorted(os.listdir(ref_dir))
    assert len(names) == 7
    for vname, defines in VARIANTS:
        copy = tmp_path / vname
        pkg = copy / "paper_2110_11392_b200"
        shutil.copytree(pkg_src, pkg, ignore=shutil.ignore_patterns("build", "*.so", "*.srchash", "__pycache__"))
        shutil.copytree(os.path.join(ROOT, "include"), copy / "include")
        build.build_debug_library(str(pkg / "libnearfield_b200.so"), defines=defines)
        # the bench-only probe library is not needed by the runner; the copy has no stale marker for it
        out = tmp_path / (vname + "_out")
        out.mkdir()
        env = dict(os.environ, PYTHONPATH=os.pathsep.join([str(copy), ROOT]))
        _run([str(out), str(copy), str(REPEATS)], env, str(copy))
        for n in names:
            a, b = np.load(ref_dir / n), np.load(out / n)
            assert a.shape == b.shape and np.array_equal(a.view(np.uint32), b.view(np.uint32)), f"{vname}: {n} differs from the default build"
