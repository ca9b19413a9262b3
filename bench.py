#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200 near-field path (contract: task prompt, section 4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

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
Multi-GPU: "replicas only": rank r runs the same config with seed r; no collective
on the data path; value = total pairs / max-over-ranks time.
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


def _ncu_traffic(config: int):
    """dram__bytes_read.sum + dram__bytes_write.sum of one k_interact launch, from the newest committed
    ``ncu --set full`` summary of this workload under profiles/ (text; None if there is none)."""
    import glob
    import re
    best = None
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", f"r*_k_interact_cfg{config}.txt"))):
        tot, n = 0.0, 0
        with open(path) as f:
            for line in f:
                m = re.match(r"dram__bytes_(read|write)\.sum\s+([0-9.]+)\s+(\w+)", line)
                if m:
                    tot += float(m.group(2)) * {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0}.get(m.group(3), 1.0)
                    n += 1
        if n == 2:
            best = (tot, os.path.relpath(path, ROOT))
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
    """oracle (as it stands) on a seeded sink-cell sample sized for ~target_s per call.
    Returns (pairs_per_s, cores, sample description, ms_per_step)."""
    import oracle
    cores = oracle.max_threads()
    ppc = cfg.N / cfg.cpd ** 3
    pairs_per_cell = ppc * ppc * (2 * cfg.R + 1) ** 3
    guess = 1.0e8 * cores                              # pairs/s, refined by the first call
    ncell = int(max(8, min(cfg.cpd ** 3, guess * min(target_s, 2.0) / pairs_per_cell)))
    t0 = time.perf_counter()
    _, pairs = oracle.accel(pos, cfg.cpd, cfg.R, cfg.eps_p, sink_cells=_sample_cells(cfg, ncell))
    dt = time.perf_counter() - t0
    # second estimate separates the fixed (binning) cost from the pair loop
    ncell2 = int(max(8, min(cfg.cpd ** 3, ncell * 3)))
    t0 = time.perf_counter()
    _, pairs2 = oracle.accel(pos, cfg.cpd, cfg.R, cfg.eps_p, sink_cells=_sample_cells(cfg, ncell2))
    dt2 = time.perf_counter() - t0
    rate = max((pairs2 - pairs) / max(dt2 - dt, 1e-3), 1e6) if pairs2 > pairs else pairs / dt
    fixed = max(dt - pairs / rate, 0.0)
    ncell3 = int(max(8, min(cfg.cpd ** 3, rate * max(target_s - fixed, 1.0) / pairs_per_cell)))
    cells = _sample_cells(cfg, ncell3)
    times, p3 = [], 0
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        _, p3 = oracle.accel(pos, cfg.cpd, cfg.R, cfg.eps_p, sink_cells=cells)
        if it >= warmup:
            times.append(time.perf_counter() - t0)
    tot = sum(times)
    sample = (f"{len(cells)} seeded random sink cells of {cfg.cpd ** 3} (all their sources), {p3:.4g} pairs per call, "
              f"wall time of the whole oracle call incl. binning all {cfg.N} particles (~{fixed:.1f} s)")
    return p3 * len(times) / tot, cores, sample, 1e3 * tot / len(times)


def bench_slabs(args, cfg, workload, dist, rank, world, local_rank, barrier):
    """N > 1, --parallel slabs: the same particle set on every rank (seed 0), each rank owns a
    pair-balanced range of x slabs; a step = halo exchange (NCCL isend/irecv) + nf_accel on own +
    ghost particles with only the own slabs as sinks.  value = all pairs / max-over-ranks time."""
    import torch
    from paper_2110_11392_b200 import slabs
    from paper_2110_11392_b200 import workloads as W
    pos_all = torch.from_numpy(W.make_positions(cfg)).cuda()
    counts = torch.bincount(slabs.cell_index(pos_all, cfg.cpd, cfg.box), minlength=cfg.cpd ** 3)
    bounds = slabs.balance_slabs(slabs.pairs_per_slab(counts, cfg.cpd, cfg.R), world)
    own, _ = slabs.local_with_ghosts(pos_all, bounds, cfg.cpd, cfg.R, rank, cfg.box)
    own = own.contiguous()
    del pos_all, counts
    snf = slabs.SlabNearField(cfg.cpd, cfg.R, cfg.eps_p, cfg.box, bounds)
    snf.nf.set_gm(1.0 / cfg.N)
    for _ in range(args.warmup):
        acc = snf.accel(own)
    torch.cuda.synchronize()
    pairs_local = snf.interaction_count()
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    l0 = snf.nf.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        acc = snf.accel(own)
    ev1.record()
    barrier()
    clocks = sampler.stop()
    launches = snf.nf.launch_count() - l0
    units, total_ms = aggregate_over_ranks(float(pairs_local) * args.steps, ev0.elapsed_time(ev1), dist)
    ok = bool(torch.isfinite(acc[:: max(1, acc.shape[0] // 100003)]).all())
    if rank == 0:
        workload = dict(workload, parallelism=f"x-slab decomposition over {world} GPUs, R-slab halo exchange per step",
                        slab_bounds=bounds)
        print(json.dumps({"metric": METRIC, "value": units / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
                          "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": workload,
                          "sink_updates_per_s": cfg.N * args.steps / (total_ms * 1e-3), "pairs_per_step": units / args.steps,
                          "clocks": clocks, "e2e": None, "gpu_launches": launches, "roofline": None, "cpu_baseline": None,
                          "ghost_particles_rank0": snf.n_ghost, "result_finite": ok}))
    dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config number 1..5 (default 4: CPD 135, N 157M)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target oracle time for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "slabs"],
                    help="N > 1: independent replicas (weak scaling, default) or ONE particle set cut into x slabs "
                         "with an R-slab halo exchange per step (strong scaling; paper_2110_11392_b200/slabs.py)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print(f"note: --warmup {args.warmup} < 3 breaks the timing rules", file=sys.stderr)

    from paper_2110_11392_b200 import workloads as W
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    base = W.CONFIGS[args.config]
    cfg = W.Config(base.name, base.cpd, base.R, base.N, base.kind, base.eps_p, base.box, seed=rank, n_spheres=base.n_spheres)
    workload = {"workload": f"BASELINE.json configs[{args.config - 1}]: {cfg.name} CPD={cfg.cpd} R={cfg.R} N={cfg.N} "
                            f"eps_p={cfg.eps_p:.6g} box=1 kind={cfg.kind} seed=rank",
                "cpd": cfg.cpd, "R": cfg.R, "N": cfg.N, "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                "l2_policy": "inputs (1.9 GB positions, ~9 GB scratch) exceed the 126 MB L2; no flush needed"
                if cfg.N * 12 > 2 * 126e6 else "L2 flushed by writing a 256 MB buffer between timed steps"}

    # ------------------------------------------------------------------ reference arm = the oracle
    if args.impl == "reference":
        if rank != 0:
            return 0
        pos = W.make_positions(cfg)
        per_step = max(4.0, min(20.0, 150.0 / max(args.steps + args.warmup, 1)))
        rate, cores, sample, ms = time_oracle(cfg, pos, per_step, steps=args.steps, warmup=args.warmup)
        line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": 0, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic", "config": workload,
                "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
                "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0,
                "note": "the reference arm is the CPU oracle (oracle/nf_oracle.c, double precision, OpenMP); "
                        "each step is a bounded sink-cell sample of the workload"}
        print(json.dumps(line))
        return 0

    # ------------------------------------------------------------------ our arm
    import torch
    from paper_2110_11392_b200.build import ensure_built
    ensure_built()                                   # no-op unless the .so is missing (fresh checkout)
    from paper_2110_11392_b200.binding import NearField, probe_pipes
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

    if args.parallel == "slabs" and world > 1:
        return bench_slabs(args, base, workload, dist, rank, world, local_rank, barrier)
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
    if not args.no_e2e:
        h_pos = torch.from_numpy(pos).pin_memory()
        h_acc = torch.empty_like(h_pos).pin_memory()
        nf.accel_host_ptr(h_pos.data_ptr(), cfg.N, h_acc.data_ptr())          # warm-up (allocates staging)
        barrier()
        t0 = time.perf_counter()
        n_e2e = max(1, min(args.steps, 3))
        for _ in range(n_e2e):
            nf.accel_host_ptr(h_pos.data_ptr(), cfg.N, h_acc.data_ptr())      # synchronous
        barrier()
        e2e_ms_local = (time.perf_counter() - t0) * 1e3
        u2, t2 = aggregate_over_ranks(float(pairs) * n_e2e, e2e_ms_local, dist)
        e2e = {"value": u2 / (t2 * 1e-3), "unit": UNIT, "h2d_bytes_per_step": cfg.N * 12, "d2h_bytes_per_step": cfg.N * 12,
               "steps": n_e2e, "ms_per_step": t2 / n_e2e, "api": "nf_accel_host (pinned host buffers)"}
        del h_pos, h_acc

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (A5): FMA-pipe issue roofline
    mp = _peaks()
    sm_max = float(mp.get("sm_max_mhz", 1965.0))
    n_sm = peaks_live["sm_count"]
    peak_lane = n_sm * 128 * sm_max * 1e6                   # FP32 FMA lanes x clock
    k_ms = statistics.mean(kernel_ms)
    traffic = _ncu_traffic(args.config)
    ach_lane = pairs * FMA_LANE_OPS_PER_PAIR / (k_ms * 1e-3)
    roofline = {"bound": "alu", "kernel": "k_interact (A5 + fused A6)",
                "achieved": ach_lane * 2 / 1e12, "peak": peak_lane * 2 / 1e12, "unit": "TFLOP/s",
                "frac": ach_lane / peak_lane, "traffic": traffic[0] if traffic else None,
                "traffic_unit": "bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum)",
                "traffic_source": traffic[1] if traffic else None,
                "convention": f"{FMA_LANE_OPS_PER_PAIR} FP32 FMA-pipe lane-ops per pair x 2 flop (SURVEY.md 8(a) note 2); "
                              f"peak = {n_sm} SMs x 128 lanes x {sm_max:.0f} MHz x 2 (derived, DESIGN.md); "
                              f"{FLOP_PER_PAIR} flop/pair convention -> {pairs * FLOP_PER_PAIR / (k_ms * 1e-3) / 1e12:.1f} TFLOP/s",
                "kernel_ms": k_ms, "kernel_share_of_step": k_ms / statistics.mean(step_ms),
                "measured_ffma_peak_lane_ops_per_s": peaks_live["ffma_lane_ops_per_s"],
                "frac_of_measured_ffma_peak": ach_lane / peaks_live["ffma_lane_ops_per_s"],
                "measured_ffma2_peak_lane_ops_per_s": peaks_live["ffma2_lane_ops_per_s"],
                "measured_mufu_rsq_lane_ops_per_s": peaks_live["mufu_rsq_lane_ops_per_s"],
                "mufu_frac": pairs / (k_ms * 1e-3) / peaks_live["mufu_rsq_lane_ops_per_s"]}

    cpu = None
    if not args.no_cpu_baseline:
        rate, cores, sample, _ = time_oracle(cfg, pos, args.cpu_seconds)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": workload,
            "sink_updates_per_s": cfg.N * world * args.steps / (total_ms * 1e-3), "pairs_per_step": pairs,
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
            "stage_ms": {k: statistics.mean(s[k] for s in stage_acc) for k in stage_acc[0]},
            "result_finite": acc_ok}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
