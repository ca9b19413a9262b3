"""Build step: compile ``csrc/*.cu`` with nvcc for sm_100a, in-tree.

``python -m paper_2110_11392_b200.build`` (or ``__graft_entry__.build()``) makes

* ``libnearfield_b200.so`` -- the product: the C ABI of ``include/nearfield.h``;
* ``libnf_pipeprobe.so``   -- a bench-only helper (``probe/nf_pipeprobe.cu``, outside ``csrc/``: the product
  library's state tag does not depend on it): FP32 / FP64 / MUFU pipe-rate microbenchmarks that give
  ``bench.py`` its live roofline denominators.  Not part of the product ABI.

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
PROBE_SRC = os.path.join(HERE, "probe", "nf_pipeprobe.cu")
SOURCES = ["nf_api.cu", "nf_binner.cu", "nf_rebin.cu", "nf_interact.cu", "nf_f64.cu", "nf_multipoles.cu", "nf_taylor.cu", "nf_step.cu",
           "nf_slabs.cu", "nf_noalloc.cu"]
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


def _probe_stale() -> bool:
    import hashlib
    with open(PROBE_SRC, "rb") as f:
        h = hashlib.sha1(f.read()).hexdigest()
    try:
        with open(PROBE_LIB + ".srchash") as f:
            return not os.path.exists(PROBE_LIB) or f.read().strip() != h
    except OSError:
        return True


def _compile_probe(verbose: bool) -> None:
    """one translation unit of its own, kept out of csrc/"""
    import hashlib
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc, *NVCC_FLAGS, "-shared", "-o", PROBE_LIB + ".tmp", PROBE_SRC]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True, stdout=sys.stderr, stderr=sys.stderr)
    os.replace(PROBE_LIB + ".tmp", PROBE_LIB)
    with open(PROBE_SRC, "rb") as f, open(PROBE_LIB + ".srchash", "w") as g:
        g.write(hashlib.sha1(f.read()).hexdigest() + "\n")


def _compile(sources: list[str], lib: str, verbose: bool) -> None:
    import hashlib
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    hh = hashlib.sha1(" ".join(NVCC_FLAGS).encode())
    for h in sorted(d for d in _deps() if d.endswith((".cuh", ".h"))):
        with open(h, "rb") as f:
            hh.update(f.read())

    def one(src: str) -> str:
        # an object is reused only if it was compiled from exactly this source, these headers and these flags:
        # the key is a content hash kept beside the .o (mtimes do not survive a copy of the tree)
        path = os.path.join(CSRC, src)
        obj = os.path.join(OBJ, src.replace(os.sep, "_") + ".o")
        k = hh.copy()
        with open(path, "rb") as f:
            k.update(f.read())
        key = k.hexdigest()
        try:
            with open(obj + ".srchash") as f:
                fresh = os.path.exists(obj) and f.read().strip() == key
        except OSError:
            fresh = False
        if not fresh:
            cmd = [nvcc, *NVCC_FLAGS, "-c", "-o", obj, path]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            subprocess.run(cmd, check=True, stdout=sys.stderr, stderr=sys.stderr)
            with open(obj + ".srchash", "w") as f:
                f.write(key + "\n")
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
    if force or _probe_stale():
        _compile_probe(verbose)
    return LIB


def build_debug_library(out: str, verbose: bool = False, defines: tuple[str, ...] = ("-DNF_DEBUG_BOUNDS",)) -> str:
    """A build of the product library with other ``defines``, written to ``out`` -- never over the in-tree library.
    Default: the -DNF_DEBUG_BOUNDS build (csrc/nf_common.cuh: every derived index is checked against the bound of
    its array; nf_sync reports a violation); tests/test_gpu_debug_bounds.py runs the small parity cases under it.
    tests/test_gpu_ring_stress.py builds the copy-ring stress variants (-DNF_NSTAGE=2 -DNF_REFILL_BELOW=1, ...)."""
    nvcc = os.environ.get("NVCC", "nvcc")
    objdir = out + ".obj"
    os.makedirs(objdir, exist_ok=True)

    def one(src: str) -> str:
        obj = os.path.join(objdir, src.replace(os.sep, "_") + ".o")
        cmd = [nvcc, *NVCC_FLAGS, *defines, "-c", "-o", obj, os.path.join(CSRC, src)]
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
    if _stale(LIB) or _probe_stale():
        build_library()
    return LIB


if __name__ == "__main__":
    if "--debug-bounds" in sys.argv:
        print(build_debug_library(sys.argv[sys.argv.index("--debug-bounds") + 1], verbose="-v" in sys.argv))
    else:
        print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
