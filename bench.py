#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200 near-field path (contract: task prompt, section 4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config all|1..5] [--impl ours|reference]

A "step" is one pass of the whole hot path (A1..A6: bin, scan, scatter, schedule, interact,
un-permute) over one synthetic particle set.  Default workload: BASELINE.json configs[3]
(CPD 135, R 2, N = 540^3 = 157 464 000, the config the north_star's roofline target names).
Metric: near-field pairwise interactions per second (pairs = sum_c n_c sum_{c' in N(c)} n_c' - N,
counted on the device by nf_interaction_count; padding and masked lanes are not work).

One JSON line on stdout (rank 0).  ``value`` = device-resident inputs; ``e2e`` = through
nf_accel_host with pinned HOST buffers (H2D + D2H inside the timed region);
``roofline`` = FMA-pipe issue roofline of the interaction kernel;
``cpu_baseline`` = the oracle timed on the host cores on a bounded sample.
``--impl reference`` times the oracle (there is no other reference implementation).
``--config all`` (the default) measures configs 1, 2, 3, 5 as well and adds them under ``per_config`` (config 4
stays the headline of the line).
Multi-GPU (N > 1): the path shards: ONE particle set is cut into pair-balanced
x slabs, one range per rank; a step = halo exchange of the R ghost slabs (isend/irecv over NCCL) +
nf_accel with the own slabs as sinks; value = all pairs / max-over-ranks time ("strong").
``--parallel replicas`` runs N independent copies instead (rank r = same config, seed r; "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "nearfield_pair_interactions_per_s"
UNIT = "pairs/s"
FMA_LANE_OPS_PER_PAIR = 14        # SURVEY.md 8(a) note 2: 14 FMA-pipe + 1 ALU + 1 MUFU per pair
FLOP_PER_PAIR = 23                # FMA = 2, rsqrt = 1, min = 1 (paper's "about 26" adds its density term)


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except OSError:
        return {}


def _library_state() -> str:
    """tag of the sources the loaded library was built from (paper_2110_11392_b200/build.py)"""
    from paper_2110_11392_b200.build import _source_hash
    return _source_hash()[:12]


def _ncu_traffic(config: int):
    """dram__bytes_read.sum + dram__bytes_write.sum of one k_interact launch, from the newest committed
    ``ncu --set full`` summary of this workload under profiles/ (text; None if there is none).
    -> (bytes, file, stale): ``stale`` unless the summary's ``# library_state:`` line names the sources
    the library in use was built from -- a capture of another kernel state is context, not this run's traffic."""
    import glob
    import re
    best = None
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", f"r*_k_interact_cfg{config}.txt"))):
        tot, n, tag = 0.0, 0, None
        with open(path) as f:
            for line in f:
                m = re.match(r"#\s*library_state:\s*(\w+)", line)
                if m:
                    tag = m.group(1)
                m = re.match(r"dram__bytes_(read|write)\.sum\s+([0-9.]+)\s+(\w+)", line)
                if m:
                    tot += float(m.group(2)) * {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0}.get(m.group(3), 1.0)
                    n += 1
        if n == 2:
            best = (tot, os.path.relpath(path, ROOT), tag != _library_state())
    return best


class ClockSampler(threading.Thread):
    """samples SM clock + throttle reasons during the timed region (pynvml, else nvidia-smi)."""

    def __init__(self, index: int, period: float = 0.1):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._halt = threading.Event()
        self._nv = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _poll_nvml(self):
        nv = self._nv
        self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
        try:
            r = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
        except Exception:
            r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake_slowdown"}
        for bit, nm in names.items():
            if r & bit:
                self.reasons.add(nm)

    def _poll_smi(self):
        import subprocess
        q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
            "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        out = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                             capture_output=True, text=True, timeout=5).stdout.strip().split(",")
        self.samples.append(float(out[0]))
        self.max_mhz = float(out[1])
        for nm, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], out[2:]):
            if v.strip().lower().startswith("active"):
                self.reasons.add(nm)

    def run(self):
        while not self._halt.is_set():
            try:
                self._poll_nvml() if self._nv else self._poll_smi()
            except Exception:
                pass
            self._halt.wait(self.period)

    def stop(self) -> dict:
        self._halt.set()
        self.join(timeout=5)
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def aggregate_over_ranks(local_units: float, local_ms: float, dist=None):
    """whole-job units and max-over-ranks time.  ``dist`` = torch.distributed (initialised) or None."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(local_units), float(local_ms)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    u = torch.tensor([local_units], dtype=torch.float64, device=dev)
    t = torch.tensor([local_ms], dtype=torch.float64, device=dev)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(u.item()), float(t.item())


def _sample_cells(cfg, n_cells: int, seed: int = 1234) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return np.sort(rng.choice(cfg.cpd ** 3, size=min(n_cells, cfg.cpd ** 3), replace=False)).astype(np.int32)


def time_oracle(cfg, pos, target_s: float, steps: int = 1, warmup: int = 0):
    """The oracle as it stands, timed so that the number does not depend on the sample size: its
    binning (all particles, one thread) is timed once on its own, and the pair loop's rate is the
    SLOPE between two seeded sink-cell samples (about 1:4), i.e. pairs added / seconds added, the
    fixed cost of each whole call cancelling.  ``steps`` repeats of the larger sample are averaged.
    -> dict for ``cpu_baseline`` (value = pair-loop pairs/s on all host cores) + ms per step."""
    import oracle
    cores = oracle.max_threads()
    ncell_all = cfg.cpd ** 3
    t0 = time.perf_counter()
    cell, _ = oracle.bin_particles(pos, cfg.cpd, cfg.box)
    oracle.cell_lists(cell, cfg.cpd)
    binning_s = time.perf_counter() - t0
    counts = np.bincount(cell, minlength=ncell_all)
    del cell

    def run(cells):
        t0 = time.perf_counter()
        _, p = oracle.accel(pos, cfg.cpd, cfg.R, cfg.eps_p, sink_cells=cells)
        return p, time.perf_counter() - t0

    ppc = cfg.N / ncell_all
    pairs_per_cell = max(ppc * ppc * (2 * cfg.R + 1) ** 3, 1.0)
    # two samples of ~target/5 and ~4 target/5 of pair-loop time (sized from a nominal 3e8 pairs/s per core;
    # the slope does not depend on that guess)
    rate0 = 3.0e8 * cores
    n1 = int(max(4, min(ncell_all, rate0 * target_s * 0.2 / pairs_per_cell)))
    n2 = int(max(8, min(ncell_all, 4 * n1)))
    c1, c2 = _sample_cells(cfg, n1, seed=12), _sample_cells(cfg, n2, seed=13)
    p1, t1 = run(c1)
    t2s, p2 = [], 0
    for it in range(warmup + steps):
        p2, t = run(c2)
        if it >= warmup:
            t2s.append(t)
    t2 = sum(t2s) / len(t2s)
    if p2 > p1 and t2 > t1:
        rate = (p2 - p1) / (t2 - t1)
        fixed = max(t1 - p1 / rate, 0.0)
    else:                                    # the whole config fits both samples (config 1): no slope to take
        rate, fixed = p2 / t2, 0.0
    full_pairs = float(np.sum(counts.astype(np.float64) * _box_filter(counts.reshape(cfg.cpd, cfg.cpd, cfg.cpd), cfg.R).ravel()) - cfg.N)
    one = _config1()
    t0 = time.perf_counter()
    _, p_one = oracle.accel(one[1], one[0].cpd, one[0].R, one[0].eps_p, nthreads=1)
    single = p_one / (time.perf_counter() - t0)
    oracle.accel(one[1], one[0].cpd, one[0].R, one[0].eps_p, nthreads=cores)            # restore the thread count
    try:
        affinity = len(os.sched_getaffinity(0))
    except AttributeError:
        affinity = os.cpu_count()
    out = {"value": rate, "unit": UNIT, "cores": cores, "affinity_cores": affinity, "kind": "oracle",
           "pair_loop_pairs_per_s": rate, "binning_s": binning_s, "fixed_s_per_call": fixed,
           "extrapolated_full_config_s": binning_s + full_pairs / rate,
           "single_thread_pairs_per_s_config1": single,
           "sample": f"slope between two seeded sink-cell samples of {len(c1)} and {len(c2)} of {ncell_all} cells (all their sources; "
                     f"{p1:.4g} and {p2:.4g} pairs, {t1:.2f} s and {t2:.2f} s per whole call); binning of all {cfg.N} particles timed "
                     f"separately ({binning_s:.2f} s, one thread); extrapolated_full_config_s = binning + all {full_pairs:.4g} pairs / slope"}
    return out, 1e3 * t2


def _config1():
    from paper_2110_11392_b200 import workloads as W
    return W.CONFIGS[1], W.make_positions(W.CONFIGS[1])


def _box_filter(n: np.ndarray, R: int) -> np.ndarray:
    """periodic (2R+1)^3 box filter of the occupancy histogram (accounting only: pair counts)"""
    f = n.astype(np.float64)
    for axis in range(3):
        acc = np.zeros_like(f)
        for sft in range(-R, R + 1):
            acc += np.roll(f, sft, axis=axis)
        f = acc
    return f


W_BASE_CPD = {1: 7, 2: 35, 3: 63, 4: 135, 5: 45}


def _workload(k: int, cfg, world: int, parallel: str) -> dict:
    par = "single GPU" if world == 1 else (f"x-slab decomposition over {world} GPUs, R-slab halo exchange per step" if parallel == "slabs"
                                           else f"replicas x{world}")
    return {"workload": f"{'BASELINE.json' if cfg.cpd == W_BASE_CPD.get(k) else 'size study, recipe of BASELINE.json'} configs[{k - 1}]: {cfg.name} CPD={cfg.cpd} R={cfg.R} N={cfg.N} "
                        f"eps_p={cfg.eps_p:.6g} box=1 kind={cfg.kind} seed={'0' if parallel == 'slabs' or world == 1 else 'rank'}",
            "cpd": cfg.cpd, "R": cfg.R, "N": cfg.N, "parallelism": par,
            "l2_policy": "inputs (1.9 GB positions, ~9 GB scratch) exceed the 126 MB L2; no flush needed"
            if cfg.N * 12 > 2 * 126e6 else "L2 flushed by writing a 256 MB buffer between timed steps"}


def _issued_ops_per_pair(nf, d_pos, cfg, pairs: int, rc_cells: float) -> float:
    """FMA-pipe lane-operations the kernel ISSUES per algorithmic pair: 11 per
    pair (3 FADD d, 3 FMA r^2, 2 FMUL rho^3, 3 FMA accumulate) in far cells and, once a close-pair
    radius is in force, everywhere; 14 (the spline polynomial as well) only in the near cells of the
    min-form regime.  Weighted by the near/far split of the pair count (accounting from the library's
    cell histogram; padding and masked lanes are not counted as work on either side)."""
    if rc_cells > 0:
        return 11.0
    n = nf.cell_histogram(d_pos).cpu().numpy().reshape(cfg.cpd, cfg.cpd, cfg.cpd)
    near_cheb = min(cfg.R, max(1, int(np.ceil(2.16 * cfg.eps_p * cfg.cpd / cfg.box))))
    near = float((n * _box_filter(n, near_cheb)).sum()) - cfg.N
    return (14.0 * near + 11.0 * (pairs - near)) / max(pairs, 1)


def measure(k: int, args, rank: int, world: int, local_rank: int, dist, barrier, seed: int, want_e2e: bool, cpu_seconds: float) -> dict:
    """one config on this rank's GPU (N = 1, or one of N replicas): the JSON fields of that workload"""
    import torch
    from paper_2110_11392_b200 import workloads as W
    from paper_2110_11392_b200.binding import NearField
    from paper_2110_11392_b200.pipeprobe import probe_pipes
    base = W.CONFIGS[k] if not getattr(args, "scale_cpd", 0) else W.scaled(W.CONFIGS[k], args.scale_cpd)
    cfg = W.Config(base.name, base.cpd, base.R, base.N, base.kind, base.eps_p, base.box, seed=seed, n_spheres=base.n_spheres)
    pos = W.make_positions(cfg)
    nf = NearField(cfg.cpd, cfg.R, cfg.eps_p, cfg.box)
    nf.set_option("stage_timing", 1)
    stream = torch.cuda.Stream()
    d_pos = torch.from_numpy(pos).cuda()
    d_acc = torch.empty_like(d_pos)
    flush = None if cfg.N * 12 > 2 * 126e6 else torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def step():
        if flush is not None:
            flush.fill_(1)
        nf.accel(d_pos, d_acc, stream=stream)

    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            step()
        stream.synchronize()
        pairs = nf.interaction_count()
        rc_cells = nf.close_radius()
        peaks_live = probe_pipes() if rank == 0 else None
        sampler = ClockSampler(local_rank)
        barrier()
        sampler.start()
        launches0 = nf.launch_count()
        kernel_ms, step_ms, stage_acc = [], [], []
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        for _ in range(args.steps):
            step()
            # per-step stage events are recorded by the library on `stream`; reading them syncs
            st = nf.stage_ms()
            stage_acc.append(st)
            kernel_ms.append(st["A5_interact_A6_unpermute"])
            step_ms.append(st["total"])
        ev1.record(stream)
        barrier()
        launches = nf.launch_count() - launches0
        clocks = sampler.stop()
    total_ms_local = sum(step_ms) if flush is not None else ev0.elapsed_time(ev1)
    units, total_ms = aggregate_over_ranks(float(pairs) * args.steps, total_ms_local, dist)
    value = units / (total_ms * 1e-3)
    nf.sync()
    acc_ok = bool(torch.isfinite(d_acc[:: max(1, cfg.N // 1000003)]).all())

    # ---- end to end through the C ABI with pinned host buffers
    e2e = None
    if want_e2e:
        h_pos = torch.from_numpy(pos).pin_memory()
        h_acc = torch.empty_like(h_pos).pin_memory()
        nf.accel_host_ptr(h_pos.data_ptr(), cfg.N, h_acc.data_ptr())          # warm-up (allocates staging)
        # the link by itself: one plain pinned copy of the same bytes each way (outside the timed region), so that the
        # reader can tell how much of e2e - value is PCIe and how much is the code
        tmp = torch.empty_like(d_pos)
        c0, c1, c2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        torch.cuda.synchronize()
        c0.record(); tmp.copy_(h_pos, non_blocking=True); c1.record(); h_acc.copy_(tmp, non_blocking=True); c2.record()
        torch.cuda.synchronize()
        h2d_ms, d2h_ms = c0.elapsed_time(c1), c1.elapsed_time(c2)
        del tmp
        barrier()
        t0 = time.perf_counter()
        n_e2e = max(1, min(args.steps, 3))
        for _ in range(n_e2e):
            nf.accel_host_ptr(h_pos.data_ptr(), cfg.N, h_acc.data_ptr())      # synchronous
        barrier()
        e2e_ms_local = (time.perf_counter() - t0) * 1e3
        u2, t2 = aggregate_over_ranks(float(pairs) * n_e2e, e2e_ms_local, dist)
        nbytes = cfg.N * 12
        e2e = {"value": u2 / (t2 * 1e-3), "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
               "steps": n_e2e, "ms_per_step": t2 / n_e2e, "api": "nf_accel_host (pinned host buffers; H2D chunks overlap the binning)",
               "pcie_GBps": {"h2d": nbytes / (h2d_ms * 1e-3) / 1e9 if h2d_ms > 0 else None, "d2h": nbytes / (d2h_ms * 1e-3) / 1e9 if d2h_ms > 0 else None},
               "plain_copy_ms": {"h2d": h2d_ms, "d2h": d2h_ms},
               "ms_over_device_step": t2 / n_e2e - total_ms / args.steps,
               "note": "the result is in input order and exists only after the kernel's fused un-permute, so the D2H copy follows the kernel "
                       "serially (ms_over_device_step ~ plain_copy_ms.d2h + what of the H2D the binning cannot hide): the link, not the code"}
        del h_pos, h_acc
    out = {"value": value, "ms_per_step": total_ms / args.steps, "config": _workload(k, cfg, world, "replicas"),
           "sink_updates_per_s": cfg.N * world * args.steps / (total_ms * 1e-3), "pairs_per_step": pairs,
           "close_pair_radius_cells": rc_cells, "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "result_finite": acc_ok}
    if rank != 0:
        nf.close()
        return out

    # ---- roofline of the dominant kernel (A5): FMA-pipe issue roofline
    mp = _peaks()
    sm_max = float(mp.get("sm_max_mhz", 1965.0))
    n_sm = peaks_live["sm_count"]
    peak_lane = n_sm * 128 * sm_max * 1e6                   # FP32 FMA lanes x clock
    k_ms = statistics.mean(kernel_ms)
    traffic = _ncu_traffic(k)
    ach_lane = pairs * FMA_LANE_OPS_PER_PAIR / (k_ms * 1e-3)
    issued = _issued_ops_per_pair(nf, d_pos, cfg, pairs, rc_cells)
    iss_lane = pairs * issued / (k_ms * 1e-3)
    out["roofline"] = {
        "bound": "alu", "kernel": "k_interact (A5 + fused A6)",
        "achieved": ach_lane * 2 / 1e12, "peak": peak_lane * 2 / 1e12, "unit": "TFLOP/s",
        "frac": ach_lane / peak_lane,
        "frac_issued": iss_lane / peak_lane, "issued_fma_lane_ops_per_pair": issued,
        "frac_issued_of_measured_ffma2_peak": iss_lane / peaks_live["ffma2_lane_ops_per_s"],
        "traffic": traffic[0] if traffic else None,
        "traffic_unit": "bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum)",
        "traffic_source": traffic[1] if traffic else None, "traffic_stale": traffic[2] if traffic else None,
        "library_state": _library_state(),
        "convention": f"frac: {FMA_LANE_OPS_PER_PAIR} FP32 FMA-pipe lane-ops per pair x 2 flop (SURVEY.md 8(a) note 2, the algorithm's count); "
                      f"frac_issued: the {issued:.2f} lane-ops per pair the kernel issues (what ncu's sm__pipe_fma_cycles_active follows); "
                      f"peak = {n_sm} SMs x 128 lanes x {sm_max:.0f} MHz x 2 (derived, DESIGN.md); "
                      f"{FLOP_PER_PAIR} flop/pair convention -> {pairs * FLOP_PER_PAIR / (k_ms * 1e-3) / 1e12:.1f} TFLOP/s",
        "kernel_ms": k_ms, "kernel_share_of_step": k_ms / statistics.mean(step_ms),
        "measured_ffma_peak_lane_ops_per_s": peaks_live["ffma_lane_ops_per_s"],
        "frac_of_measured_ffma_peak": ach_lane / peaks_live["ffma_lane_ops_per_s"],
        "measured_ffma2_peak_lane_ops_per_s": peaks_live["ffma2_lane_ops_per_s"],
        "measured_mufu_rsq_lane_ops_per_s": peaks_live["mufu_rsq_lane_ops_per_s"],
        "measured_dfma_lane_ops_per_s": peaks_live["dfma_lane_ops_per_s"],
        "mufu_frac": pairs / (k_ms * 1e-3) / peaks_live["mufu_rsq_lane_ops_per_s"]}
    out["stage_ms"] = {kk: statistics.mean(st[kk] for st in stage_acc) for kk in stage_acc[0]}
    if args.neighbours:
        out["neighbour_steps"] = _neighbour_steps(nf, d_pos, d_acc, cfg, peaks_live)
    nf.close()
    del d_pos, d_acc
    torch.cuda.empty_cache()
    out["cpu_baseline"] = None
    if cpu_seconds > 0:
        out["cpu_baseline"], _ = time_oracle(cfg, pos, cpu_seconds)
    return out


def _neighbour_steps(nf, d_pos, d_acc, cfg, peaks_live, order: int = 8) -> dict:
    """device times of the pipeline steps either side of NearForce at this workload (Table 1:
    TaylorForce, Kick, Drift, multipoles in Finish), each on a pinned binning (nf_bin) so that the
    sort is timed once on its own; FP64 kernels against the measured DFMA rate."""
    import torch
    cml = (order + 3) * (order + 2) * (order + 1) // 6

    def timed(fn, reps=3):
        fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    res = {"order": order}
    nf.unbin()
    res["bin_ms"] = timed(lambda: nf.bin(d_pos))
    M = nf.multipoles(d_pos, order)
    res["multipoles_ms"] = timed(lambda: nf.multipoles(d_pos, order))
    res["taylor_ms"] = timed(lambda: nf.taylor_accel(d_pos, M, order, acc=d_acc))
    del M
    vel = torch.zeros_like(d_pos)
    res["kick_drift_ms"] = timed(lambda: nf.kick_drift(d_pos, vel, d_acc, 0.0, 0.0))
    res["timestep_ratio_ms"] = timed(lambda: nf.timestep_ratio(d_pos, vel, d_acc))          # Eq. 1's per-cell reduction (on the pinned binning; syncs)
    # nf_rebin after a drift of 0.05 cell rms per component (a few per cent of the particles change cell: PAPER.md:356
    # "most particles stay in their cell") against the full sort above; the drift itself is not timed
    vel = torch.randn_like(d_pos) * (0.05 * cfg.box / cfg.cpd)
    nf.bin(d_pos)
    ts = []
    for _ in range(3):
        nf.kick_drift(d_pos, vel, d_acc, 0.0, 1.0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        nf.rebin(d_pos)
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    res["rebin_ms_after_drift_0.05_cell"] = min(ts[1:])          # the first call allocates the insert list
    del vel
    nf.unbin()
    dfma = peaks_live["dfma_lane_ops_per_s"]
    # algorithmic FP64 FMA-class operations per particle: multipoles cml FMAs + (p+1)(p+2)/2
    # products + 3p powers; Taylor ~4 per coefficient (Horner value + derivative, two folds)
    mp_ops = cml + (order + 1) * (order + 2) // 2 + 3 * order
    ty_ops = 4 * cml
    res["multipoles_frac_of_dfma_peak"] = cfg.N * mp_ops / (res["multipoles_ms"] * 1e-3) / dfma
    res["taylor_frac_of_dfma_peak"] = cfg.N * ty_ops / (res["taylor_ms"] * 1e-3) / dfma
    res["multipoles_particles_per_s"] = cfg.N / (res["multipoles_ms"] * 1e-3)
    res["taylor_particles_per_s"] = cfg.N / (res["taylor_ms"] * 1e-3)
    res["kick_drift_GBps"] = cfg.N * 12 * 5 / (res["kick_drift_ms"] * 1e-3) / 1e9      # read pos, vel, acc; write pos, vel
    res["bin_GBps_algorithmic"] = cfg.N * 72 / (res["bin_ms"] * 1e-3) / 1e9             # 72 B per particle
    return res


def bench_slabs(args, k, dist, rank, world, local_rank, barrier) -> dict:
    """ONE particle set (seed 0, every rank generates it and keeps its own slabs) over `world` GPUs: a
    step = halo exchange of the R ghost slabs (isend/irecv: NCCL over NVLink) + nf_accel on own + ghost
    particles with only the own slabs as sinks.  value = all pairs / max-over-ranks time (strong scaling)."""
    import torch
    from paper_2110_11392_b200 import slabs
    from paper_2110_11392_b200 import workloads as W
    from paper_2110_11392_b200.binding import NearField
    from paper_2110_11392_b200.pipeprobe import probe_pipes
    cfg = W.CONFIGS[k]
    pos_np = W.make_positions(cfg)
    with NearField(cfg.cpd, cfg.R, cfg.eps_p, cfg.box) as planner:
        pos_all = torch.from_numpy(pos_np).cuda()
        bounds = slabs.plan_slabs(planner, pos_all, world)           # same input on every rank: no all_reduce needed, same cuts
        x0, nx = bounds[rank]
        buf = torch.empty_like(pos_all)
        n_own = planner.select_slabs(pos_all, x0, nx, out=buf)
        own = buf[:n_own].clone()
        del buf, pos_all
    del pos_np
    torch.cuda.empty_cache()
    snf = slabs.SlabNearField(cfg.cpd, cfg.R, cfg.eps_p, cfg.box, bounds, gm=1.0 / cfg.N)
    snf.nf.set_option("stage_timing", 1)
    for _ in range(args.warmup):
        acc = snf.accel(own, validate=True)
    torch.cuda.synchronize()
    pairs_local = snf.interaction_count()
    rc_cells = snf.nf.close_radius()
    peaks_live = probe_pipes() if rank == 0 else None
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    l0 = snf.nf.launch_count()
    kernel_ms = []
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        acc = snf.accel(own)
        kernel_ms.append(snf.nf.stage_ms()["A5_interact_A6_unpermute"])
    ev1.record()
    barrier()
    clocks = sampler.stop()
    launches = snf.nf.launch_count() - l0
    units, total_ms = aggregate_over_ranks(float(pairs_local) * args.steps, ev0.elapsed_time(ev1), dist)
    ok = bool(torch.isfinite(acc[:: max(1, acc.shape[0] // 100003)]).all())

    # end to end: own particles from pinned host memory each step, accelerations back to pinned host memory
    e2e = None
    if not args.no_e2e:
        h_own = own.cpu().pin_memory()
        h_acc = torch.empty_like(h_own).pin_memory()
        d_own = torch.empty_like(own)
        barrier()
        t0 = time.perf_counter()
        n_e2e = max(1, min(args.steps, 3))
        for _ in range(n_e2e):
            d_own.copy_(h_own, non_blocking=True)
            h_acc.copy_(snf.accel(d_own), non_blocking=True)
            torch.cuda.synchronize()
        barrier()
        u2, t2 = aggregate_over_ranks(float(pairs_local) * n_e2e, (time.perf_counter() - t0) * 1e3, dist)
        e2e = {"value": u2 / (t2 * 1e-3), "unit": UNIT, "h2d_bytes_per_step": n_own * 12, "d2h_bytes_per_step": n_own * 12,
               "steps": n_e2e, "ms_per_step": t2 / n_e2e,
               "api": "pinned host -> device copy of the rank's particles, SlabNearField.accel (halo exchange + nf_accel), result to pinned host; bytes are rank 0's"}
    out = {"value": units / (total_ms * 1e-3), "ms_per_step": total_ms / args.steps, "config": dict(_workload(k, cfg, world, "slabs"), slab_bounds=bounds),
           "sink_updates_per_s": cfg.N * args.steps / (total_ms * 1e-3), "pairs_per_step": units / args.steps,
           "close_pair_radius_cells": rc_cells, "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "result_finite": ok,
           "halo_bytes_per_step_rank0": snf.halo_bytes, "ghost_particles_rank0": snf.n_ghost, "own_particles_rank0": n_own}
    if rank == 0:
        mp = _peaks()
        sm_max = float(mp.get("sm_max_mhz", 1965.0))
        peak_lane = peaks_live["sm_count"] * 128 * sm_max * 1e6
        k_ms = statistics.mean(kernel_ms)
        ach = pairs_local * FMA_LANE_OPS_PER_PAIR / (k_ms * 1e-3)
        issued = 11.0 if rc_cells > 0 else float("nan")
        out["roofline"] = {"bound": "alu", "kernel": "k_interact (A5 + fused A6) on rank 0", "achieved": ach * 2 / 1e12, "peak": peak_lane * 2 / 1e12,
                           "unit": "TFLOP/s", "frac": ach / peak_lane, "frac_issued": pairs_local * issued / (k_ms * 1e-3) / peak_lane,
                           "issued_fma_lane_ops_per_pair": issued, "traffic": None, "kernel_ms": k_ms,
                           "kernel_share_of_step": k_ms / (total_ms / args.steps), "pairs_rank0": pairs_local,
                           "convention": f"{FMA_LANE_OPS_PER_PAIR} FP32 FMA-pipe lane-ops per pair x 2 flop; peak = SMs x 128 lanes x {sm_max:.0f} MHz x 2 of ONE GPU"}
        out["cpu_baseline"] = None                     # timed on rank 0 at N = 1 only
    snf.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="all", help="'all' (default): BASELINE.json config 4 (CPD 135, N 157M) as the headline of the line plus "
                                                    "configs 1, 2, 3, 5 under per_config; or one config number 1..5")
    ap.add_argument("--scale-cpd", type=int, default=0, help="with --config K: run config K's RECIPE (particles per cell, distribution, "
                    "softening rule) on a grid of this many cells per dimension instead of its own -- a size study, not a BASELINE.json workload "
                    "(e.g. --config 2 --scale-cpd 100: 40 per cell, 40 M particles)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target pair-loop time of the oracle for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--neighbours", action="store_true", help="also time nf_bin / nf_multipoles / nf_taylor_accel / nf_kick_drift at the workload")
    ap.add_argument("--parallel", default=None, choices=["slabs", "replicas"],
                    help="N > 1: ONE particle set cut into x slabs with an R-slab halo exchange per step (default; strong "
                         "scaling; paper_2110_11392_b200/slabs.py), or independent replicas (weak scaling).  Given explicitly, "
                         "'slabs' also runs the sharded code path on one GPU (one range, no ghosts)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print(f"note: --warmup {args.warmup} < 3 breaks the timing rules", file=sys.stderr)

    from paper_2110_11392_b200 import workloads as W
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    want_all = args.config == "all" and not args.scale_cpd
    if args.scale_cpd and args.config == "all":
        raise SystemExit("bench.py: --scale-cpd needs --config K")
    k_main = 4 if want_all else int(args.config)
    slabs_mode = (world > 1 and args.parallel != "replicas") or args.parallel == "slabs"

    # ------------------------------------------------------------------ reference arm = the oracle
    if args.impl == "reference":
        if rank != 0:
            return 0
        cfg = W.CONFIGS[k_main]
        pos = W.make_positions(cfg)
        per_step = max(4.0, min(20.0, 120.0 / max(args.steps + args.warmup, 1)))
        cpu, ms = time_oracle(cfg, pos, per_step, steps=args.steps, warmup=args.warmup)
        line = {"impl": "reference", "metric": METRIC, "value": cpu["value"], "unit": UNIT, "n_gpus": 0, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong" if slabs_mode else "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": _workload(k_main, cfg, 1, "replicas"),
                "cpu_baseline": cpu,
                "e2e": {"value": cpu["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0,
                "note": "the reference arm is the CPU oracle (oracle/nf_oracle.c, double precision, OpenMP); value = its pair-loop "
                        "rate (slope between two sink-cell samples, the same quantity as our arm's cpu_baseline.value); each step is "
                        "one whole oracle call on the larger sample (ms_per_step)"}
        print(json.dumps(line))
        return 0

    # ------------------------------------------------------------------ our arm
    import torch
    from paper_2110_11392_b200.build import ensure_built
    ensure_built()                                   # no-op unless the libraries are missing or older than their sources
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    cpu_s = 0.0 if (args.no_cpu_baseline or world > 1) else args.cpu_seconds
    if slabs_mode:
        res = bench_slabs(args, k_main, dist, rank, world, local_rank, barrier)
        scaling = "strong"
    else:
        res = measure(k_main, args, rank, world, local_rank, dist, barrier, seed=rank, want_e2e=not args.no_e2e, cpu_seconds=cpu_s)
        scaling = "weak"
    per_config = None
    if want_all and not slabs_mode:
        per_config = {}
        for k in (1, 2, 3, 5):
            r = measure(k, args, rank, world, local_rank, dist, barrier, seed=rank, want_e2e=not args.no_e2e,
                        cpu_seconds=min(cpu_s, 6.0))
            if rank == 0:
                per_config[str(k)] = r
    if rank == 0:
        line = {"metric": METRIC, "value": res.pop("value"), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": res.pop("ms_per_step"), "higher_is_better": True, "scaling": scaling, "vs_baseline": None,
                "dtype": "f32", "data": "synthetic"}
        line.update(res)
        if per_config is not None:
            line["per_config"] = per_config
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
