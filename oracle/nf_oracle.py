"""ctypes loader for ``nf_oracle.c`` (TEST INFRASTRUCTURE -- see the C file's header).

The shared object is built with gcc on first use (``-O3 -march=native -fopenmp``, no
``-ffast-math``) and named after a hash of the source and of the host CPU's flags, so a copy
built on another machine is never loaded by mistake.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nf_oracle.c")
_lib = None


def _cpu_tag() -> str:
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    with open(_SRC, "rb") as f:
        src = f.read()
    return hashlib.sha1(src + flags.encode()).hexdigest()[:12]


def lib_path() -> str:
    return os.path.join(_HERE, f"libnf_oracle.{_cpu_tag()}.so")


def build(force: bool = False) -> str:
    """Compile ``nf_oracle.c`` with gcc (building the checker is not using it)."""
    out = lib_path()
    if force or not os.path.exists(out):
        tmp = out + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-std=c99", "-shared", "-fPIC",
               "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True, stdout=sys.stderr, stderr=sys.stderr)
        os.replace(tmp, out)
    return out


def _load():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        i64, i32, dbl, vp = ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_void_p
        L.nfo_max_threads.restype = i32
        L.nfo_force_factor.restype = dbl
        L.nfo_force_factor.argtypes = [dbl, dbl]
        L.nfo_plummer_factor.restype = dbl
        L.nfo_plummer_factor.argtypes = [dbl, dbl]
        L.nfo_bin.restype = i32
        L.nfo_bin.argtypes = [vp, i64, i32, dbl, vp, vp]
        L.nfo_cell_lists.restype = None
        L.nfo_cell_lists.argtypes = [vp, i64, i64, vp, vp]
        L.nfo_neighbors.restype = None
        L.nfo_neighbors.argtypes = [i32, i32, i32, vp, vp]
        L.nfo_pair_count.restype = i64
        L.nfo_pair_count.argtypes = [vp, i32, i32]
        L.nfo_accel.restype = i64
        L.nfo_accel.argtypes = [vp, i64, i32, i32, dbl, dbl, dbl, vp, i64, vp, i32]
        L.nfo_kick_drift.restype = None
        L.nfo_kick_drift.argtypes = [vp, vp, vp, i64, dbl, dbl, dbl]
        L.nfo_timestep_ratio.restype = i32
        L.nfo_timestep_ratio.argtypes = [vp, vp, vp, i64, i32, dbl, vp]
        L.nfo_taylor_accel.restype = i32
        L.nfo_taylor_accel.argtypes = [vp, i64, i32, dbl, i32, vp, vp]
        L.nfo_multipoles.restype = i32
        L.nfo_multipoles.argtypes = [vp, i64, i32, dbl, i32, vp]
        L.nfo_accel_variant.restype = i64
        L.nfo_accel_variant.argtypes = [vp, i64, i32, i32, dbl, dbl, dbl, i32, dbl, vp, i64, vp, vp, i32]
        _lib = L
    return _lib


def _f32pos(pos) -> np.ndarray:
    p = np.ascontiguousarray(pos, dtype=np.float32)
    if p.ndim != 2 or p.shape[1] != 3:
        raise ValueError("pos must be [N,3]")
    return p


def max_threads() -> int:
    return int(_load().nfo_max_threads())


def force_factor(r: float, eps_s: float) -> float:
    """f with F = f * r_vec, Eq. 3."""
    return float(_load().nfo_force_factor(float(r), float(eps_s)))


def plummer_factor(r: float, eps_p: float) -> float:
    """f with F = f * r_vec, Eq. 2."""
    return float(_load().nfo_plummer_factor(float(r), float(eps_p)))


def bin_particles(pos, cpd: int, box: float = 1.0):
    """-> (cell[N] int32, off[N,3] float64 offsets from cell centres, box units)."""
    p = _f32pos(pos)
    N = p.shape[0]
    cell = np.empty(N, dtype=np.int32)
    off = np.empty((N, 3), dtype=np.float64)
    rc = _load().nfo_bin(p.ctypes.data, N, cpd, float(box), cell.ctypes.data, off.ctypes.data)
    if rc != 0:
        raise ValueError("non-finite position")
    return cell, off


def cell_lists(cell: np.ndarray, cpd: int):
    """-> (offsets[cpd^3+1] int64, order[N] int64): grid order, stable within a cell."""
    cell = np.ascontiguousarray(cell, dtype=np.int32)
    ncell = cpd ** 3
    offsets = np.empty(ncell + 1, dtype=np.int64)
    order = np.empty(cell.shape[0], dtype=np.int64)
    _load().nfo_cell_lists(cell.ctypes.data, cell.shape[0], ncell, offsets.ctypes.data, order.ctypes.data)
    return offsets, order


def neighbors(cpd: int, R: int, cellid: int):
    """-> (ids[(2R+1)^3] int32, image[(2R+1)^3,3] int8), (a,b,c) lexicographic."""
    nn = (2 * R + 1) ** 3
    ids = np.empty(nn, dtype=np.int32)
    img = np.empty((nn, 3), dtype=np.int8)
    _load().nfo_neighbors(cpd, R, int(cellid), ids.ctypes.data, img.ctypes.data)
    return ids, img


def pair_count(offsets: np.ndarray, cpd: int, R: int) -> int:
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    return int(_load().nfo_pair_count(offsets.ctypes.data, cpd, R))


def accel(pos, cpd: int, R: int, eps_p: float, box: float = 1.0, gm: float | None = None,
          sink_cells=None, nthreads: int = 0):
    """Near-field accelerations by the definition.  -> (acc[N,3] float64, pairs evaluated).

    ``sink_cells``: optional int32 array of cell ids; only particles in those cells are
    evaluated (the rest of ``acc`` stays 0).  ``gm`` defaults to 1/N."""
    p = _f32pos(pos)
    N = p.shape[0]
    if gm is None:
        gm = 1.0 / max(N, 1)
    acc = np.zeros((N, 3), dtype=np.float64)
    if sink_cells is None:
        sc_ptr, nsc = None, 0
    else:
        sc = np.ascontiguousarray(sink_cells, dtype=np.int32)
        sc_ptr, nsc = sc.ctypes.data, sc.shape[0]
    pairs = _load().nfo_accel(p.ctypes.data, N, cpd, R, float(eps_p), float(box), float(gm),
                              sc_ptr, nsc, acc.ctypes.data, int(nthreads))
    if pairs < 0:
        raise ValueError("nfo_accel: bad arguments or non-finite position")
    return acc, int(pairs)


def accel_variant(pos, cpd: int, R: int, eps_p: float, box: float = 1.0, gm: float | None = None,
                  law: str = "spline", density_b: float = 0.0, sink_cells=None, nthreads: int = 0):
    """The build-time variants of the paper's kernel, by the definition:
    ``law`` = "spline" (Eq. 3), "plummer" (Eq. 2) or "newton" (no softening,
    PAPER.md:218: r/|r|^3, coincident pairs contribute 0; eps_p ignored); ``density_b`` > 0 adds the
    FoF-scale density estimate sum_{q != p, r < b} (b^2 - r^2).
    -> (acc[N,3] float64, dens[N] float64 or None, pairs visited)."""
    p = _f32pos(pos)
    N = p.shape[0]
    if gm is None:
        gm = 1.0 / max(N, 1)
    acc = np.zeros((N, 3), dtype=np.float64)
    dens = np.zeros(N, dtype=np.float64) if density_b > 0 else None
    if sink_cells is None:
        sc_ptr, nsc = None, 0
    else:
        sc = np.ascontiguousarray(sink_cells, dtype=np.int32)
        sc_ptr, nsc = sc.ctypes.data, sc.shape[0]
    pairs = _load().nfo_accel_variant(p.ctypes.data, N, cpd, R, float(eps_p), float(box), float(gm),
                                      {"spline": 0, "plummer": 1, "newton": 2}[law], float(density_b), sc_ptr, nsc,
                                      acc.ctypes.data, dens.ctypes.data if dens is not None else None, int(nthreads))
    if pairs < 0:
        raise ValueError("nfo_accel_variant: bad arguments or non-finite position")
    return acc, dens, int(pairs)


def multipoles(pos, cpd: int, order: int = 8, box: float = 1.0) -> np.ndarray:
    """Cell multipoles of Eq. 4 in the complete basis -> float64 [cpd^3, cml],
    cml = (p+3)(p+2)(p+1)/6, index order = the (a, b, c) nesting of the paper's pseudo-code."""
    p = _f32pos(pos)
    cml = (order + 3) * (order + 2) * (order + 1) // 6
    M = np.zeros((cpd ** 3, cml), dtype=np.float64)
    rc = _load().nfo_multipoles(p.ctypes.data, p.shape[0], cpd, float(box), int(order), M.ctypes.data)
    if rc != cml:
        raise ValueError("nfo_multipoles: bad arguments or non-finite position")
    return M


def multipole_index(order: int):
    """the (a, b, c) triple of every column of ``multipoles`` (the pseudo-code's nesting order)"""
    return [(a, b, c) for a in range(order + 1) for b in range(order - a + 1) for c in range(order - a - b + 1)]


def kick_drift(pos, vel, acc, dt_kick: float, dt_drift: float, box: float = 1.0):
    """Kick then Drift of the KDK leapfrog (Table 1 :379-380) on float32 state.
    -> (new pos, new vel) float32 [N,3]; the inputs are not modified."""
    p = _f32pos(pos).copy()
    v = np.ascontiguousarray(vel, dtype=np.float32).copy()
    a = np.ascontiguousarray(acc, dtype=np.float32)
    _load().nfo_kick_drift(p.ctypes.data, v.ctypes.data, a.ctypes.data, p.shape[0], float(dt_kick), float(dt_drift), float(box))
    return p, v


def timestep_ratio(pos, vel, acc, cpd: int, box: float = 1.0) -> np.ndarray:
    """particle part of Eq. 1: [min_c v_rms/a_max, global v_rms/a_max, v_rms,global, a_max,global]"""
    p = _f32pos(pos)
    v = np.ascontiguousarray(vel, dtype=np.float32)
    a = np.ascontiguousarray(acc, dtype=np.float32)
    out = np.zeros(4, dtype=np.float64)
    if _load().nfo_timestep_ratio(p.ctypes.data, v.ctypes.data, a.ctypes.data, p.shape[0], cpd, float(box), out.ctypes.data) != 0:
        raise ValueError("nfo_timestep_ratio: bad arguments or non-finite position")
    return out


def taylor_accel(pos, T, cpd: int, order: int = 8, box: float = 1.0) -> np.ndarray:
    """Far-field acceleration -grad phi from per-cell Taylor coefficients of the potential in the
    complete basis (reading F1).  T: [cpd^3, cml] float64 -> acc float64 [N,3]."""
    p = _f32pos(pos)
    cml = (order + 3) * (order + 2) * (order + 1) // 6
    T = np.ascontiguousarray(T, dtype=np.float64)
    if T.shape != (cpd ** 3, cml):
        raise ValueError(f"T must have shape {(cpd ** 3, cml)}")
    acc = np.zeros((p.shape[0], 3), dtype=np.float64)
    if _load().nfo_taylor_accel(p.ctypes.data, p.shape[0], cpd, float(box), int(order), T.ctypes.data, acc.ctypes.data) != 0:
        raise ValueError("nfo_taylor_accel: bad arguments or non-finite position")
    return acc
