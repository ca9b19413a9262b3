"""Thin ctypes binding of ``include/nearfield.h`` -- argument marshalling only.

Every step of the path runs in the CUDA kernels of ``libnearfield_b200.so``; there is no CPU
fallback.  If the library is missing this module raises at import (build it with
``python -m paper_2110_11392_b200.build``).  PyTorch supplies device memory and streams.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
NF_OK, NF_EINVAL, NF_ECUDA, NF_ENOMEM, NF_EPOS = 0, 1, 2, 3, 4
_STATUS = {0: "NF_OK", 1: "NF_EINVAL", 2: "NF_ECUDA", 3: "NF_ENOMEM", 4: "NF_EPOS"}
NF_N_STAGES = 8
STAGE_NAMES = ["A1_key_hist", "A2_scan", "A3_scatter_rank_gather", "A4_scheduler",
               "A5_interact_A6_unpermute", "total", "reserved6", "reserved7"]

# every symbol include/nearfield.h declares
SYMBOLS = ["nf_create", "nf_destroy", "nf_set_gm", "nf_accel", "nf_accel_host", "nf_sync",
           "nf_last_error", "nf_set_option", "nf_stage_ms", "nf_debug_cells", "nf_debug_neighbors",
           "nf_interaction_count", "nf_debug_read", "nf_launch_count", "nf_close_radius",
           "nf_set_softening", "nf_set_density_radius", "nf_accel4", "nf_set_sink_slabs", "nf_accel_f64", "nf_multipoles", "nf_kick_drift", "nf_timestep_ratio", "nf_taylor_accel",
           "nf_debug_delivered_pairs", "nf_bounds_checked", "nf_bin", "nf_rebin", "nf_unbin", "nf_cell_histogram", "nf_slab_pairs", "nf_select_slabs",
           "nf_cell_offsets_noalloc", "nf_cell_offsets_noalloc_error"]


class NearFieldError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


def lib_path() -> str:
    """the in-tree library"""
    return os.path.join(_HERE, "libnearfield_b200.so")


def load_library() -> ctypes.CDLL:
    path = lib_path()
    if not os.path.exists(path):
        raise ImportError(f"{path} is not built (python -m paper_2110_11392_b200.build); "
                          "there is no CPU fallback")
    L = ctypes.CDLL(path)
    vp, i64, i32, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
    L.nf_create.restype = i32
    L.nf_create.argtypes = [ctypes.POINTER(vp), i32, i32, dbl, dbl]
    L.nf_destroy.restype = i32
    L.nf_destroy.argtypes = [vp]
    L.nf_set_gm.restype = i32
    L.nf_set_gm.argtypes = [vp, dbl]
    L.nf_accel.restype = i32
    L.nf_accel.argtypes = [vp, vp, i64, vp, vp]
    L.nf_accel4.restype = i32
    L.nf_accel4.argtypes = [vp, vp, i64, vp, vp]
    L.nf_set_softening.restype = i32
    L.nf_set_softening.argtypes = [vp, i32]
    L.nf_kick_drift.restype = i32
    L.nf_kick_drift.argtypes = [vp, vp, vp, vp, i64, dbl, dbl, vp]
    L.nf_timestep_ratio.restype = i32
    L.nf_timestep_ratio.argtypes = [vp, vp, vp, vp, i64, vp, vp]
    L.nf_taylor_accel.restype = i32
    L.nf_taylor_accel.argtypes = [vp, vp, i64, i32, vp, vp, i32, vp]
    L.nf_multipoles.restype = i32
    L.nf_multipoles.argtypes = [vp, vp, i64, i32, vp, vp]
    L.nf_accel_f64.restype = i32
    L.nf_accel_f64.argtypes = [vp, vp, i64, vp, vp]
    L.nf_set_sink_slabs.restype = i32
    L.nf_set_sink_slabs.argtypes = [vp, i32, i32]
    L.nf_set_density_radius.restype = i32
    L.nf_set_density_radius.argtypes = [vp, dbl]
    L.nf_accel_host.restype = i32
    L.nf_accel_host.argtypes = [vp, vp, i64, vp]
    L.nf_sync.restype = i32
    L.nf_sync.argtypes = [vp]
    L.nf_last_error.restype = ctypes.c_char_p
    L.nf_last_error.argtypes = [vp]
    L.nf_set_option.restype = i32
    L.nf_set_option.argtypes = [vp, ctypes.c_char_p, dbl]
    L.nf_stage_ms.restype = i32
    L.nf_stage_ms.argtypes = [vp, vp]
    L.nf_debug_cells.restype = i32
    L.nf_debug_cells.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(vp),
                                 ctypes.POINTER(vp), ctypes.POINTER(i64)]
    L.nf_debug_neighbors.restype = i32
    L.nf_debug_neighbors.argtypes = [vp, i32, vp, vp]
    L.nf_interaction_count.restype = i32
    L.nf_interaction_count.argtypes = [vp, ctypes.POINTER(i64)]
    L.nf_debug_delivered_pairs.restype = i32
    L.nf_debug_delivered_pairs.argtypes = [vp, vp]
    L.nf_bin.restype = i32
    L.nf_bin.argtypes = [vp, vp, i64, vp]
    L.nf_rebin.restype = i32
    L.nf_rebin.argtypes = [vp, vp, i64, vp]
    L.nf_unbin.restype = i32
    L.nf_unbin.argtypes = [vp]
    L.nf_cell_histogram.restype = i32
    L.nf_cell_histogram.argtypes = [vp, vp, i64, vp, vp]
    L.nf_slab_pairs.restype = i32
    L.nf_slab_pairs.argtypes = [vp, vp, vp, vp, vp]
    L.nf_select_slabs.restype = i32
    L.nf_select_slabs.argtypes = [vp, vp, i64, i32, i32, vp, ctypes.POINTER(i64), vp]
    L.nf_close_radius.restype = i32
    L.nf_close_radius.argtypes = [vp, ctypes.POINTER(dbl)]
    L.nf_bounds_checked.restype = i32
    L.nf_bounds_checked.argtypes = []
    L.nf_launch_count.restype = i32
    L.nf_launch_count.argtypes = [vp, ctypes.POINTER(i64)]
    L.nf_debug_read.restype = i32
    L.nf_debug_read.argtypes = [vp, vp, vp, ctypes.c_uint64]
    L.nf_cell_offsets_noalloc.restype = i32
    L.nf_cell_offsets_noalloc.argtypes = [vp, i64, vp, vp]
    L.nf_cell_offsets_noalloc_error.restype = ctypes.c_char_p
    L.nf_cell_offsets_noalloc_error.argtypes = []
    return L


_L = load_library()


def bounds_checked() -> bool:
    """nf_bounds_checked: is the loaded library the -DNF_DEBUG_BOUNDS build?"""
    return bool(_L.nf_bounds_checked())


NF_NOALLOC_MAX_CELLS = 8388608


def cell_offsets_noalloc(counts, offsets=None, stream=None):
    """nf_cell_offsets_noalloc: exclusive scan of a cell histogram (CUDA int32 [ncell]) into ``offsets`` (CUDA int32 /
    uint32 storage, [ncell + 1]) with no context and no device allocation inside the library -- for callers that
    cannot let a library call cudaMalloc (a code whose own pool holds the whole GPU; a loop whose overlapping streams
    a cudaMalloc would stall).  Pass ``offsets`` yourself to keep the call free of any allocation: when it is None
    this wrapper -- not the library -- makes the tensor with torch.  The tensors' device must be the current device.
    At most NF_NOALLOC_MAX_CELLS cells; calls that may overlap on the GPU race on the shared scratch (see nearfield.h)."""
    import torch
    if not (counts.is_cuda and counts.dtype == torch.int32 and counts.is_contiguous() and counts.dim() == 1):
        raise ValueError("counts must be a contiguous 1-D CUDA int32 tensor")
    n = counts.numel()
    if offsets is None:
        offsets = torch.empty(n + 1, dtype=torch.int32, device=counts.device)
    elif not (offsets.is_cuda and offsets.dtype == torch.int32 and offsets.is_contiguous() and offsets.numel() == n + 1
              and offsets.device == counts.device):
        raise ValueError("offsets must be a contiguous CUDA int32 tensor of ncell + 1 entries on counts' device")
    st = torch.cuda.current_stream(counts.device) if stream is None else stream
    rc = _L.nf_cell_offsets_noalloc(counts.data_ptr() if n else None, n, offsets.data_ptr(), ctypes.c_void_p(st.cuda_stream))
    if rc != NF_OK:
        raise NearFieldError(rc, _L.nf_cell_offsets_noalloc_error().decode())
    return offsets


class NearField:
    """nf_create / nf_accel / nf_destroy with torch tensors (or host numpy arrays) as buffers."""

    def __init__(self, cpd: int, R: int, eps_plummer: float, box: float = 1.0):
        self._h = ctypes.c_void_p()
        rc = _L.nf_create(ctypes.byref(self._h), int(cpd), int(R), float(eps_plummer), float(box))
        if rc != NF_OK:
            raise NearFieldError(rc, _L.nf_last_error(None).decode())
        self.cpd, self.R, self.eps_plummer, self.box = int(cpd), int(R), float(eps_plummer), float(box)
        self._N = 0
        self._pinned = None          # the tensor nf_bin / nf_rebin pinned (kept alive: the pin is keyed on its address)

    # -- helpers
    def _check(self, rc: int):
        if rc != NF_OK:
            raise NearFieldError(rc, _L.nf_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            _L.nf_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- the path
    def set_gm(self, gm: float):
        self._check(_L.nf_set_gm(self._h, float(gm)))

    def set_option(self, name: str, value: float):
        self._check(_L.nf_set_option(self._h, name.encode(), float(value)))

    def accel(self, pos, acc=None, stream=None):
        """pos: CUDA float32 tensor [N,3] (contiguous).  Returns acc [N,3] on the same device.
        Enqueued on ``stream`` (default: torch's current stream); not synchronised."""
        import torch
        if not (pos.is_cuda and pos.dtype == torch.float32 and pos.is_contiguous() and pos.dim() == 2 and pos.shape[1] == 3):
            raise ValueError("pos must be a contiguous CUDA float32 tensor of shape [N,3]")
        N = pos.shape[0]
        if acc is None:
            acc = torch.empty_like(pos)
        elif not (acc.is_cuda and acc.dtype == torch.float32 and acc.is_contiguous() and acc.shape == pos.shape):
            raise ValueError("acc must match pos")
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        self._N = N
        self._check(_L.nf_accel(self._h, pos.data_ptr() if N else None, N, acc.data_ptr() if N else None,
                                ctypes.c_void_p(st.cuda_stream)))
        return acc

    def set_softening(self, law: str):
        """"spline" (Eq. 3, default), "plummer" (Eq. 2) or "newton" (no softening) -- nf_set_softening"""
        self._check(_L.nf_set_softening(self._h, {"spline": 0, "plummer": 1, "newton": 2}[law]))

    def bin(self, pos, stream=None):
        """nf_bin: sort ``pos`` into grid order now and keep the binning for the following calls on ``pos``.
        The library recognises the pinned buffer by its address and length alone.  This wrapper therefore keeps a
        reference to ``pos`` while it is pinned, so that torch's caching allocator cannot hand the same address to a
        new tensor of the same size (which would silently be served the old grid order).  Changing ``pos`` in place
        by anything but ``kick_drift`` is still the caller's to announce: ``unbin()`` or ``bin()`` again."""
        import torch
        if not (pos.is_cuda and pos.dtype == torch.float32 and pos.is_contiguous() and pos.dim() == 2 and pos.shape[1] == 3):
            raise ValueError("pos must be a contiguous CUDA float32 tensor of shape [N,3]")
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        self._N = pos.shape[0]
        self._check(_L.nf_bin(self._h, pos.data_ptr(), pos.shape[0], ctypes.c_void_p(st.cuda_stream)))
        self._pinned = pos

    def rebin(self, pos, stream=None):
        """nf_rebin: update the kept grid order after the particles moved (insert list + merge) and pin it."""
        import torch
        if not (pos.is_cuda and pos.dtype == torch.float32 and pos.is_contiguous() and pos.dim() == 2 and pos.shape[1] == 3):
            raise ValueError("pos must be a contiguous CUDA float32 tensor of shape [N,3]")
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        self._N = pos.shape[0]
        self._check(_L.nf_rebin(self._h, pos.data_ptr(), pos.shape[0], ctypes.c_void_p(st.cuda_stream)))
        self._pinned = pos

    def unbin(self):
        self._check(_L.nf_unbin(self._h))
        self._pinned = None

    def delivered_pairs(self):
        """nf_debug_delivered_pairs -> (deliveries incl. self meetings, self meetings) of the last accel."""
        out = (ctypes.c_int64 * 2)()
        self._check(_L.nf_debug_delivered_pairs(self._h, out))
        return int(out[0]), int(out[1])

    def set_sink_slabs(self, x0: int, nx: int):
        """only particles in x slabs [x0, x0 + nx) (periodic) are sinks -- nf_set_sink_slabs"""
        self._check(_L.nf_set_sink_slabs(self._h, int(x0), int(nx)))

    def cell_histogram(self, pos, stream=None):
        """nf_cell_histogram -> int32 [cpd^3] on the device (summable across ranks with all_reduce)."""
        import torch
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        counts = torch.empty(self.cpd ** 3, dtype=torch.int32, device=pos.device)
        N = pos.shape[0]
        self._check(_L.nf_cell_histogram(self._h, pos.data_ptr() if N else None, N, counts.data_ptr(), ctypes.c_void_p(st.cuda_stream)))
        return counts

    def slab_pairs(self, counts, stream=None):
        """nf_slab_pairs -> (pairs int64 [cpd], particles int64 [cpd]) per x slab, on the device."""
        import torch
        if not (counts.is_cuda and counts.dtype == torch.int32 and counts.is_contiguous() and counts.numel() == self.cpd ** 3):
            raise ValueError("counts must be a contiguous CUDA int32 tensor of cpd^3 entries")
        st = torch.cuda.current_stream(counts.device) if stream is None else stream
        pairs = torch.empty(self.cpd, dtype=torch.int64, device=counts.device)
        npart = torch.empty(self.cpd, dtype=torch.int64, device=counts.device)
        self._check(_L.nf_slab_pairs(self._h, counts.data_ptr(), pairs.data_ptr(), npart.data_ptr(), ctypes.c_void_p(st.cuda_stream)))
        return pairs, npart

    def select_slabs(self, pos, x0: int, nx: int, out=None, stream=None) -> int:
        """nf_select_slabs: particles of ``pos`` in x slabs [x0, x0+nx) (periodic) -> first rows of ``out``
        ([>=count, 3] CUDA float32, input order kept); returns the count.  ``out`` None: count only."""
        import torch
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        N = pos.shape[0]
        if out is not None and not (out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and out.numel() >= 3 * N):
            raise ValueError("out must be a contiguous CUDA float32 tensor with room for all of pos")
        n = ctypes.c_int64()
        self._check(_L.nf_select_slabs(self._h, pos.data_ptr() if N else None, N, int(x0), int(nx),
                                       out.data_ptr() if out is not None else None, ctypes.byref(n), ctypes.c_void_p(st.cuda_stream)))
        return int(n.value)

    def set_density_radius(self, b: float):
        self._check(_L.nf_set_density_radius(self._h, float(b)))

    def accel4(self, pos, acc4=None, stream=None):
        """nf_accel4: -> [N,4] (ax, ay, az, density estimate of PAPER.md:256)."""
        import torch
        if not (pos.is_cuda and pos.dtype == torch.float32 and pos.is_contiguous() and pos.dim() == 2 and pos.shape[1] == 3):
            raise ValueError("pos must be a contiguous CUDA float32 tensor of shape [N,3]")
        N = pos.shape[0]
        if acc4 is None:
            acc4 = torch.zeros((N, 4), dtype=torch.float32, device=pos.device)
        elif not (acc4.is_cuda and acc4.dtype == torch.float32 and acc4.is_contiguous() and tuple(acc4.shape) == (N, 4)):
            raise ValueError("acc4 must be a contiguous CUDA float32 tensor of shape [N,4]")
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        self._N = N
        self._check(_L.nf_accel4(self._h, pos.data_ptr() if N else None, N, acc4.data_ptr() if N else None,
                                 ctypes.c_void_p(st.cuda_stream)))
        return acc4

    def accel_f64(self, pos, stream=None):
        """nf_accel_f64: the double-precision direct sum on the GPU -> float64 [N,3]."""
        import torch
        if not (pos.is_cuda and pos.dtype == torch.float32 and pos.is_contiguous() and pos.dim() == 2 and pos.shape[1] == 3):
            raise ValueError("pos must be a contiguous CUDA float32 tensor of shape [N,3]")
        N = pos.shape[0]
        acc = torch.zeros((N, 3), dtype=torch.float64, device=pos.device)
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        self._N = N
        self._check(_L.nf_accel_f64(self._h, pos.data_ptr() if N else None, N, acc.data_ptr() if N else None,
                                    ctypes.c_void_p(st.cuda_stream)))
        return acc

    def multipoles(self, pos, order: int = 8, stream=None):
        """nf_multipoles: Eq. 4 in the complete basis -> float64 [cpd^3, (p+3)(p+2)(p+1)/6] on the device."""
        import torch
        if not (pos.is_cuda and pos.dtype == torch.float32 and pos.is_contiguous() and pos.dim() == 2 and pos.shape[1] == 3):
            raise ValueError("pos must be a contiguous CUDA float32 tensor of shape [N,3]")
        N = pos.shape[0]
        cml = (order + 3) * (order + 2) * (order + 1) // 6
        M = torch.empty((self.cpd ** 3, max(cml, 1)), dtype=torch.float64, device=pos.device)
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        self._N = N
        self._check(_L.nf_multipoles(self._h, pos.data_ptr() if N else None, N, int(order), M.data_ptr(),
                                     ctypes.c_void_p(st.cuda_stream)))
        return M

    def taylor_accel(self, pos, T, order: int = 8, acc=None, accumulate: bool = False, stream=None):
        """nf_taylor_accel: T float64 [cpd^3, cml] on the device -> acc float32 [N,3] (written or added to)."""
        import torch
        N = pos.shape[0]
        cml = (order + 3) * (order + 2) * (order + 1) // 6
        if not (T.is_cuda and T.dtype == torch.float64 and T.is_contiguous() and tuple(T.shape) == (self.cpd ** 3, cml)):
            raise ValueError(f"T must be a contiguous CUDA float64 tensor of shape {(self.cpd ** 3, cml)}")
        if acc is None:
            acc = torch.zeros_like(pos)
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        self._N = N
        self._check(_L.nf_taylor_accel(self._h, pos.data_ptr() if N else None, N, int(order), T.data_ptr(),
                                       acc.data_ptr() if N else None, 1 if accumulate else 0, ctypes.c_void_p(st.cuda_stream)))
        return acc

    def kick_drift(self, pos, vel, acc, dt_kick: float, dt_drift: float, stream=None):
        """nf_kick_drift: in place on CUDA float32 [N,3] tensors pos and vel."""
        import torch
        for t in (pos, vel, acc):
            if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.shape == pos.shape):
                raise ValueError("pos, vel, acc must be contiguous CUDA float32 tensors of the same shape [N,3]")
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        N = pos.shape[0]
        self._check(_L.nf_kick_drift(self._h, pos.data_ptr() if N else None, vel.data_ptr() if N else None,
                                     acc.data_ptr() if N else None, N, float(dt_kick), float(dt_drift), ctypes.c_void_p(st.cuda_stream)))

    def timestep_ratio(self, pos, vel, acc, stream=None) -> np.ndarray:
        """nf_timestep_ratio -> [min_c v_rms/a_max, global ratio, v_rms,global, a_max,global] (synchronises)."""
        import torch
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        N = pos.shape[0]
        self._N = N
        out = np.zeros(4, dtype=np.float64)
        self._check(_L.nf_timestep_ratio(self._h, pos.data_ptr() if N else None, vel.data_ptr() if N else None,
                                         acc.data_ptr() if N else None, N, out.ctypes.data, ctypes.c_void_p(st.cuda_stream)))
        return out

    def accel_ptr(self, d_pos: int, N: int, d_acc: int, cuda_stream: int = 0):
        """raw-pointer form of nf_accel (used by tests of the error paths)."""
        self._N = N
        self._check(_L.nf_accel(self._h, ctypes.c_void_p(d_pos), int(N), ctypes.c_void_p(d_acc), ctypes.c_void_p(cuda_stream)))

    def accel_host(self, h_pos: np.ndarray, h_acc: np.ndarray | None = None) -> np.ndarray:
        """nf_accel_host: host float32 [N,3] in, host float32 [N,3] out; synchronous."""
        h_pos = np.ascontiguousarray(h_pos, dtype=np.float32)
        if h_acc is None:
            h_acc = np.empty_like(h_pos)
        self._N = h_pos.shape[0]
        self._check(_L.nf_accel_host(self._h, h_pos.ctypes.data, h_pos.shape[0], h_acc.ctypes.data))
        return h_acc

    def accel_host_ptr(self, h_pos_ptr: int, N: int, h_acc_ptr: int):
        self._N = N
        self._check(_L.nf_accel_host(self._h, ctypes.c_void_p(h_pos_ptr), int(N), ctypes.c_void_p(h_acc_ptr)))

    def sync(self):
        self._check(_L.nf_sync(self._h))

    def stage_ms(self) -> dict:
        buf = (ctypes.c_float * NF_N_STAGES)()
        self._check(_L.nf_stage_ms(self._h, buf))
        return {STAGE_NAMES[i]: float(buf[i]) for i in range(6)}

    def close_radius(self) -> float:
        v = ctypes.c_double()
        self._check(_L.nf_close_radius(self._h, ctypes.byref(v)))
        return float(v.value)

    def launch_count(self) -> int:
        v = ctypes.c_int64()
        self._check(_L.nf_launch_count(self._h, ctypes.byref(v)))
        return int(v.value)

    def interaction_count(self) -> int:
        v = ctypes.c_int64()
        self._check(_L.nf_interaction_count(self._h, ctypes.byref(v)))
        return int(v.value)

    def debug_neighbors(self, cell: int):
        nn = (2 * self.R + 1) ** 3
        ids = np.empty(nn, dtype=np.int32)
        img = np.empty((nn, 3), dtype=np.int8)
        self._check(_L.nf_debug_neighbors(self._h, int(cell), ids.ctypes.data, img.ctypes.data))
        return ids, img

    def debug_cells(self):
        """-> dict of host numpy copies: offsets[cpd^3+1], perm[N], poffsets[cpd^3+1],
        sorted_xyz[Npad,3] (cell units), sorted_key[Npad] (high bit = padding slot)."""
        self.sync()
        p_off, p_perm, p_sorted, p_poff = (ctypes.c_void_p() for _ in range(4))
        stride = ctypes.c_int64()
        self._check(_L.nf_debug_cells(self._h, ctypes.byref(p_off), ctypes.byref(p_perm), ctypes.byref(p_sorted),
                                      ctypes.byref(p_poff), ctypes.byref(stride)))
        ncell = self.cpd ** 3

        def d2h(ptr, count, dtype):
            out = np.empty(count, dtype=dtype)
            if count:
                self._check(_L.nf_debug_read(self._h, ctypes.c_void_p(ptr), out.ctypes.data, out.nbytes))
            return out

        offsets = d2h(p_off.value, ncell + 1, np.uint32)
        poff = d2h(p_poff.value, ncell + 1, np.uint32)
        perm = d2h(p_perm.value, self._N, np.uint32)
        npad, st = int(poff[-1]), int(stride.value)
        planes = [d2h(p_sorted.value + 4 * st * k, npad, np.float32 if k < 3 else np.uint32) for k in range(4)]
        return {"offsets": offsets, "perm": perm, "poffsets": poff,
                "sorted_xyz": np.stack(planes[:3], -1), "sorted_key": planes[3]}
