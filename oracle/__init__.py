"""CPU oracle for the Abacus near-field force -- TEST INFRASTRUCTURE, not product code.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with the CUDA path and
does not import ``paper_2110_11392_b200``.  See ``nf_oracle.c`` for the definition it follows
(PAPER.md:132 Eq. 3, :143, :218) and the list of pins.
"""
from .nf_oracle import (accel, accel_variant, bin_particles, build, cell_lists, force_factor, max_threads,
                        neighbors, pair_count, plummer_factor, lib_path, multipoles, multipole_index, kick_drift, timestep_ratio, taylor_accel)

__all__ = ["accel", "accel_variant", "bin_particles", "build", "cell_lists", "force_factor", "max_threads",
           "neighbors", "pair_count", "plummer_factor", "lib_path", "multipoles", "multipole_index", "kick_drift", "timestep_ratio", "taylor_accel"]
