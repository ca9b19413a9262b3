"""The small parity cases under the -DNF_DEBUG_BOUNDS build of the library (csrc/nf_common.cuh: every index the
kernels derive from the offset tables, the ring cursor, the sink order and the permutations is checked against
the bound of its array; nf_sync reports a violation).  compute-sanitizer is not available on this pool, so this
is the memory-safety evidence for the ring / cursor / lock machinery of the interaction kernel and for the binner.

The debug library is built into a COPY of the package under tmp_path (never over the in-tree library) and the
cases run in a subprocess whose PYTHONPATH puts that copy first."""
import os
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r'''
import numpy as np, torch
import paper_2110_11392_b200.binding as B
from paper_2110_11392_b200 import workloads as W
import oracle
torch.manual_seed(0)
assert B.bounds_checked(), "not the NF_DEBUG_BOUNDS build"
assert B.lib_path().startswith(r"%(copy)s"), B.lib_path()

def check(got, ref, label):
    d = np.linalg.norm(got - ref, axis=1); a = np.linalg.norm(ref, axis=1)
    rms = np.sqrt((a ** 2).mean())
    assert d.max() <= 1e-5 * rms, (label, d.max() / rms)

CASES = [("cfg1", W.CONFIGS[1], {}), ("cfg2@13", W.scaled(W.CONFIGS[2], 13), {}), ("cfg3@10", W.scaled(W.CONFIGS[3], 10), {}),
         ("cfg4@9", W.scaled(W.CONFIGS[4], 9), {}), ("cfg5@9 R3", W.scaled(W.CONFIGS[5], 9), {}), ("cfg2@5 = 2R+1", W.scaled(W.CONFIGS[2], 5), {}),
         ("min form R2 eps .1 cell", W.Config("m2", 7, 2, 30 * 7 ** 3, "uniform", 0.1 / 7, seed=32), {"rc_cells": 0.0}), ("cfg3@10 rc .2", W.scaled(W.CONFIGS[3], 10), {"rc_cells": 0.2}),
         ("R4", W.Config("r4", 9, 4, 30 * 9 ** 3, "uniform", 1.0 / (30 * 9 ** 3) ** (1 / 3) / 40, seed=8), {}),
         ("sparse", W.Config("s", 16, 2, 2 * 16 ** 3, "uniform", 1.0 / (2 * 16 ** 3) ** (1 / 3) / 40, seed=9), {})]
for label, cfg, opts in CASES:
    pos = W.make_positions(cfg)
    ref, _ = oracle.accel(pos, cfg.cpd, cfg.R, cfg.eps_p)
    with B.NearField(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        for k, v in opts.items():
            nf.set_option(k, v)
        d = torch.from_numpy(pos).cuda()
        got = nf.accel(d); nf.sync()                                  # nf_sync raises on a failed bounds check
        check(got.cpu().numpy().astype(np.float64), ref, label)
        nf.delivered_pairs(); nf.sync()                               # the counting instantiation walks the same ring
        nf.set_density_radius(0.35 * cfg.cell); nf.accel4(d); nf.sync()
        nf.set_softening("plummer"); nf.accel(d); nf.sync()
        nf.set_softening("newton"); nf.accel(d); nf.sync()
        moved = torch.remainder(d + 0.01 * torch.rand_like(d), 1.0).contiguous()
        moved[moved >= 1.0] = 0.0
        nf.bin(d); nf.rebin(moved); nf.multipoles(moved, 8); nf.sync()
# a heavy cell (long-cell ranking, chunked stages) next to odd and empty cells
rng = np.random.default_rng(8)
pos = np.concatenate([((2 + rng.random((9001, 3))) / 6), ((np.array([3, 2, 2]) + rng.random((37, 3))) / 6), ((np.array([5, 5, 0]) + rng.random((5, 3))) / 6)]).astype(np.float32)
ref, _ = oracle.accel(pos, 6, 2, 0.001)
with B.NearField(6, 2, 0.001, 1.0) as nf:
    got = nf.accel(torch.from_numpy(pos).cuda()); nf.sync()
    check(got.cpu().numpy().astype(np.float64), ref, "heavy cell")
    h = nf.accel_host(pos); nf.sync()
print("BOUNDS-OK")
'''


@pytest.mark.gpu
def test_small_parity_cases_under_the_bounds_checked_build(tmp_path):
    from paper_2110_11392_b200 import build
    pkg_src = os.path.dirname(os.path.abspath(build.__file__))
    copy = tmp_path / "dbg"
    pkg = copy / "paper_2110_11392_b200"
    shutil.copytree(pkg_src, pkg, ignore=shutil.ignore_patterns("build", "*.so", "*.srchash", "__pycache__"))
    shutil.copytree(os.path.join(ROOT, "include"), copy / "include")
    build.build_debug_library(str(pkg / "libnearfield_b200.so"))
    env = dict(os.environ, PYTHONPATH=os.pathsep.join([str(copy), ROOT]))
    r = subprocess.run([sys.executable, "-c", SCRIPT % {"copy": str(copy)}], cwd=str(copy), env=env, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0 and "BOUNDS-OK" in r.stdout, r.stdout[-2000:] + r.stderr[-4000:]
