"""Host-side logic of bench.py: rank aggregation over gloo (world_size 2), the oracle timing
leg on a tiny config, and the JSON contract of the reference arm."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r'''
import os, sys, json
sys.path.insert(0, os.environ["NF_ROOT"])
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
r = dist.get_rank()
units, ms = bench.aggregate_over_ranks(100.0 * (r + 1), 10.0 + 5.0 * r, dist)
if r == 0:
    print(json.dumps({"units": units, "ms": ms, "world": dist.get_world_size()}))
dist.destroy_process_group()
'''


def test_aggregate_over_two_gloo_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    env = dict(os.environ, NF_ROOT=ROOT)
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29731", str(script)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    r = json.loads(line)
    assert r == {"units": 300.0, "ms": 15.0, "world": 2}       # sum of units, max of times


def test_aggregate_single_rank():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(7.0, 3.0, None) == (7.0, 3.0)


def test_oracle_timing_leg_and_sampling():
    sys.path.insert(0, ROOT)
    import bench
    from paper_2110_11392_b200 import workloads as W
    cfg = W.scaled(W.CONFIGS[2], 9)
    pos = W.make_positions(cfg)
    cells = bench._sample_cells(cfg, 50)
    assert len(cells) == 50 and len(set(cells.tolist())) == 50 and cells.max() < 9 ** 3
    assert np.array_equal(cells, bench._sample_cells(cfg, 50))
    cpu, ms = bench.time_oracle(cfg, pos, 0.5)
    assert cpu["value"] > 1e6 and cpu["cores"] >= 1 and "sink-cell samples" in cpu["sample"] and ms > 0
    assert cpu["value"] == cpu["pair_loop_pairs_per_s"] and cpu["binning_s"] > 0 and cpu["affinity_cores"] >= 1
    assert cpu["single_thread_pairs_per_s_config1"] > 1e6 and cpu["extrapolated_full_config_s"] > 0
    # the slope does not depend on the sample size: twice the budget gives the same rate within timing noise
    cpu2, _ = bench.time_oracle(cfg, pos, 1.0)
    assert 0.5 < cpu2["value"] / cpu["value"] < 2.0


def test_reference_arm_json_contract():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    r = json.loads(out.stdout.strip().splitlines()[-1])
    assert r["impl"] == "reference" and r["unit"] == "pairs/s" and r["value"] > 0
    assert r["metric"] == "nearfield_pair_interactions_per_s" and r["higher_is_better"] is True
    assert r["cpu_baseline"]["kind"] == "oracle" and r["cpu_baseline"]["cores"] >= 1
    assert r["cpu_baseline"]["value"] == r["value"] and "binning_s" in r["cpu_baseline"]
    assert r["e2e"]["h2d_bytes_per_step"] == 0 and r["e2e"]["value"] == r["value"]
    assert "workload" in r["config"]
