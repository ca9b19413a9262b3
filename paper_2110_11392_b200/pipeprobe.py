"""Loader of ``libnf_pipeprobe.so`` -- a bench-only helper, not part of the product's C ABI.

``probe_pipes()`` runs the pipe-rate microbenchmarks of ``probe/nf_pipeprobe.cu`` on the current
CUDA device; ``bench.py`` prints them as the live roofline denominators beside the derived peak.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))


def probe_pipes() -> dict:
    path = os.path.join(_HERE, "libnf_pipeprobe.so")
    if not os.path.exists(path):
        raise ImportError(f"{path} is not built (python -m paper_2110_11392_b200.build)")
    L = ctypes.CDLL(path)
    L.nfp_probe_pipes.restype = ctypes.c_int
    L.nfp_probe_pipes.argtypes = [ctypes.c_void_p]
    out = (ctypes.c_double * 6)()
    rc = L.nfp_probe_pipes(out)
    if rc != 0:
        raise RuntimeError(f"nfp_probe_pipes failed with status {rc}")
    return {"ffma_lane_ops_per_s": out[0], "ffma2_lane_ops_per_s": out[1], "mufu_rsq_lane_ops_per_s": out[2],
            "sm_count": int(out[3]), "sm_clock_mhz": out[4], "dfma_lane_ops_per_s": out[5]}
