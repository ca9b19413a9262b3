"""Build step: compile ``csrc/*.cu`` with nvcc for sm_100a, in-tree.

``python -m paper_2110_11392_b200.build`` (or ``__graft_entry__.build()``) makes

* ``libnearfield_b200.so`` -- the product: the C ABI of ``include/nearfield.h``;
* ``libnf_pipeprobe.so``   -- a bench-only helper (``csrc/probe/nf_pipeprobe.cu``): FP32 / FP64 / MUFU
  pipe-rate microbenchmarks that give ``bench.py`` its live roofline denominators.  Not part of the
  product ABI.
* ``libnf_opbench.so``     -- a bench-only helper (``microbench/nf_opbench.cu``): the register-operand and
  trip-loop-replica microbenchmarks behind DESIGN.md section 6 (``python -m paper_2110_11392_b200.opbench``).

nvcc cross-compiles without a GPU.  The .so files are git-ignored but travel with the repo snapshot.
Translation units are compiled in parallel and linked once.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libnearfield_b200.so")
PROBE_LIB = os.path.join(HERE, "libnf_pipeprobe.so")
OPBENCH_LIB = os.path.join(HERE, "libnf_opbench.so")
OPBENCH_SRC = os.path.join(HERE, "microbench", "nf_opbench.cu")
SOURCES = ["nf_api.cu", "nf_binner.cu", "nf_rebin.cu", "nf_interact.cu", "nf_f64.cu", "nf_multipoles.cu", "nf_taylor.cu", "nf_step.cu",
           "nf_slabs.cu", "nf_noalloc.cu"]
PROBE_SOURCES = [os.path.join("probe", "nf_pipeprobe.cu")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-Wno-format-truncation"]


def _deps() -> list[str]:
    d = []
    for root, _, files in os.walk(CSRC):
        d += [os.path.join(root, f) for f in files]
    return d + [os.path.join(HERE, "..", "include", "nearfield.h")]


def _source_hash() -> str:
    """content hash of every source and header (mtimes do not survive a copy of the tree)"""
    import hashlib
    h = hashlib.sha1()
    for d in sorted(_deps()):
        h.update(os.path.relpath(d, HERE).encode())
        with open(d, "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def _stale(lib: str) -> bool:
    """missing, or built from other sources than the ones in the tree now"""
    try:
        with open(lib + ".srchash") as f:
            return not os.path.exists(lib) or f.read().strip() != _source_hash()
    except OSError:
        return True


def _opbench_stale() -> bool:
    import hashlib
    with open(OPBENCH_SRC, "rb") as f:
        h = hashlib.sha1(f.read()).hexdigest()
    try:
        with open(OPBENCH_LIB + ".srchash") as f:
            return not os.path.exists(OPBENCH_LIB) or f.read().strip() != h
    except OSError:
        return True


def _compile_opbench(verbose: bool) -> None:
    """one translation unit of its own (kept out of csrc/: the product library's state tag does not depend on it)"""
    import hashlib
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc, *NVCC_FLAGS, "-shared", "-o", OPBENCH_LIB + ".tmp", OPBENCH_SRC]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True, stdout=sys.stderr, stderr=sys.stderr)
    os.replace(OPBENCH_LIB + ".tmp", OPBENCH_LIB)
    with open(OPBENCH_SRC, "rb") as f, open(OPBENCH_LIB + ".srchash", "w") as g:
        g.write(hashlib.sha1(f.read()).hexdigest() + "\n")


def _compile(sources: list[str], lib: str, verbose: bool) -> None:
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    headers = [d for d in _deps() if d.endswith((".cuh", ".h"))]
    newest_header = max(os.path.getmtime(h) for h in headers)

    def one(src: str) -> str:
        path = os.path.join(CSRC, src)
        obj = os.path.join(OBJ, src.replace(os.sep, "_") + ".o")
        if not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(path), newest_header):
            cmd = [nvcc, *NVCC_FLAGS, "-c", "-o", obj, path]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            subprocess.run(cmd, check=True, stdout=sys.stderr, stderr=sys.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=min(8, len(sources))) as ex:
        objs = list(ex.map(one, sources))
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", lib + ".tmp", *objs],
                   check=True, stdout=sys.stderr, stderr=sys.stderr)
    os.replace(lib + ".tmp", lib)
    with open(lib + ".srchash", "w") as f:
        f.write(_source_hash() + "\n")


def build_library(force: bool = False, verbose: bool = False) -> str:
    """Compile both libraries if a source or header is newer than them (or ``force``)."""
    if force:
        for f in os.listdir(OBJ) if os.path.isdir(OBJ) else []:
            os.remove(os.path.join(OBJ, f))
    if force or _stale(LIB):
        _compile(SOURCES, LIB, verbose)
    if force or _stale(PROBE_LIB):
        _compile(PROBE_SOURCES, PROBE_LIB, verbose)
    if force or _opbench_stale():
        _compile_opbench(verbose)
    return LIB


def build_debug_library(out: str, verbose: bool = False) -> str:
    """The -DNF_DEBUG_BOUNDS build of the product library (csrc/nf_common.cuh: every derived index is checked
    against the bound of its array; nf_sync reports a violation), written to ``out`` -- never over the
    in-tree library.  tests/test_gpu_debug_bounds.py runs the small parity cases under it."""
    nvcc = os.environ.get("NVCC", "nvcc")
    objdir = out + ".obj"
    os.makedirs(objdir, exist_ok=True)

    def one(src: str) -> str:
        obj = os.path.join(objdir, src.replace(os.sep, "_") + ".o")
        cmd = [nvcc, *NVCC_FLAGS, "-DNF_DEBUG_BOUNDS", "-c", "-o", obj, os.path.join(CSRC, src)]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.run(cmd, check=True, stdout=sys.stderr, stderr=sys.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=min(8, len(SOURCES))) as ex:
        objs = list(ex.map(one, SOURCES))
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", out, *objs],
                   check=True, stdout=sys.stderr, stderr=sys.stderr)
    return out


def ensure_built() -> str:
    """Make sure the in-tree libraries exist and are not older than their sources (a fresh checkout
    has none: they are not tracked).  A build step, not a fallback: without nvcc a stale or missing
    library raises instead of being loaded silently."""
    if _stale(LIB) or _stale(PROBE_LIB) or _opbench_stale():
        build_library()
    return LIB


if __name__ == "__main__":
    if "--debug-bounds" in sys.argv:
        print(build_debug_library(sys.argv[sys.argv.index("--debug-bounds") + 1], verbose="-v" in sys.argv))
    else:
        print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
