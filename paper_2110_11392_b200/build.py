"""Build step: compile ``csrc/*.cu`` into ``libnearfield_b200.so`` in-tree with nvcc for sm_100a.

``python -m paper_2110_11392_b200.build`` (or ``__graft_entry__.build()``).  nvcc
cross-compiles without a GPU.  The .so is git-ignored but travels with the repo snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libnearfield_b200.so")
SOURCES = ["nf_api.cu", "nf_binner.cu", "nf_interact.cu", "nf_f64.cu", "nf_multipoles.cu", "nf_taylor.cu", "nf_step.cu", "nf_probe.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-Xcompiler", "-Wno-format-truncation"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "nearfield.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build_library(force: bool = False, verbose: bool = False, out: str | None = None, defines: tuple = ()) -> str:
    """Compile the library.  ``out`` / ``defines`` build a tuning variant (-DNAME=VALUE for the
    knobs of csrc/nf_common.cuh) somewhere else; the default build is the product."""
    lib = out or LIB
    if force or out is not None or _stale():
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc, *NVCC_FLAGS, *[f"-D{d}" for d in defines], "-o", lib + ".tmp", *[os.path.join(CSRC, s) for s in SOURCES]]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.run(cmd, check=True, stdout=sys.stderr, stderr=sys.stderr)
        os.replace(lib + ".tmp", lib)
    return lib


def ensure_built() -> str:
    """Build the library only if the .so is missing (a fresh checkout: the .so is not tracked).
    A build step, not a fallback: without nvcc this raises."""
    return LIB if os.path.exists(LIB) else build_library(force=True)


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
