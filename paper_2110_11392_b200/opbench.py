"""Loader of ``libnf_opbench.so`` -- a bench-only helper, not part of the product's C ABI.

``python -m paper_2110_11392_b200.opbench`` runs the microbenchmarks of ``microbench/nf_opbench.cu`` on the
current CUDA device and prints one JSON object: how many cycles one warp-instruction holds a scheduler's
pipe as a function of its VARYING 64-bit register operands (packed f32x2, scalar FFMA, DFMA), and a replica
of the interaction kernel's trip loop with the pair arithmetic all packed / accumulates scalar / all scalar
(DESIGN.md section 6).  ``bench.py`` adds the same object to its line as ``roofline.operand_probe``.
"""
from __future__ import annotations

import ctypes
import json
import os

_HERE = os.path.dirname(os.path.abspath(__file__))


def _clock_mhz() -> float:
    try:
        with open(os.path.join(_HERE, "..", "MEASURED_PEAKS.json")) as f:
            return float(json.load(f).get("sm_max_mhz", 1965.0))
    except OSError:
        return 1965.0


def operand_probe(clock_mhz: float | None = None) -> dict:
    path = os.path.join(_HERE, "libnf_opbench.so")
    if not os.path.exists(path):
        raise ImportError(f"{path} is not built (python -m paper_2110_11392_b200.build)")
    L = ctypes.CDLL(path)
    L.nfo_opbench.restype = ctypes.c_int
    L.nfo_opbench.argtypes = [ctypes.c_double, ctypes.c_void_p]
    out = (ctypes.c_double * 17)()
    clk = clock_mhz or _clock_mhz()
    rc = L.nfo_opbench(clk, out)
    if rc != 0:
        raise RuntimeError(f"nfo_opbench failed with status {rc}")
    r = [round(float(v), 3) for v in out[:14]]
    return {"clock_mhz": clk, "geometry": "4 CTAs x 128 threads per SM (the interaction kernel's occupancy), 8 independent chains per thread",
            "cycles_per_warp_instruction_per_scheduler": {
                "ffma2_1_varying_reg_operand": r[0], "ffma2_2_varying": r[1], "ffma2_3_varying_accumulate": r[2],
                "fadd2_1_varying_plus_broadcast_scalar": r[3], "fadd2_2_varying": r[4], "fmul2_1_varying": r[5], "fmul2_2_varying": r[6],
                "ffma_scalar_3_varying": r[7], "dfma_1_varying": r[8], "dfma_2_varying_accumulate": r[9], "dfma_3_varying": r[10]},
            "trip_loop_replica": {"cycles_per_trip_of_16_pairs": {"all_packed": r[11], "accumulates_scalar": r[12], "all_scalar": r[13]},
                                  "pairs_per_s": {"all_packed": float(out[14]), "accumulates_scalar": float(out[15]), "all_scalar": float(out[16])},
                                  "ideal_cycles_if_every_packed_instruction_took_2": 176}}


if __name__ == "__main__":
    print(json.dumps(operand_probe()))
