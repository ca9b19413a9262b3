"""x-slab decomposition (paper_2110_11392_b200/slabs.py): host logic on CPU, the halo exchange
over gloo with world_size 2, and (GPU) a decomposition emulated rank by rank on one device
against the single-call result and the oracle."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest
import torch

from paper_2110_11392_b200 import slabs
from paper_2110_11392_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ----------------------------------------------------------------------------- host logic (CPU)
def oracle_select(oracle_mod, pos: torch.Tensor, cpd: int):
    """a ``select(x0, nx)`` over ``pos`` from the ORACLE's binning (tests only; the product's comes
    from nf_select_slabs)"""
    cell, _ = oracle_mod.bin_particles(pos.numpy(), cpd)
    xs = torch.from_numpy(cell // (cpd * cpd))
    return (lambda x0, nx: pos[torch.remainder(xs - x0, cpd) < nx]), xs


def test_slab_runs_cover_exactly():
    assert slabs.slab_runs([3, 4, 5], 9) == [(3, 3)]
    assert sorted(slabs.slab_runs([8, 0, 1, 4], 9)) == [(4, 1), (8, 3)]
    assert slabs.slab_runs([], 9) == []
    for cpd, ss in ((5, [0, 1, 2, 3, 4]), (7, [6, 0]), (7, [1, 3, 5])):
        got = [(x0 + i) % cpd for x0, n in slabs.slab_runs(ss, cpd) for i in range(n)]
        assert sorted(got) == sorted(ss)


@pytest.mark.parametrize("world", [1, 2, 3, 4, 8])
def test_balance_slabs_covers_and_balances(world):
    rng = np.random.default_rng(world)
    work = torch.from_numpy(rng.integers(1, 1000, size=35))
    b = slabs.balance_slabs(work, world)
    assert len(b) == world and b[0][0] == 0 and sum(nx for _, nx in b) == 35 and all(nx >= 1 for _, nx in b)
    for (x0, nx), (x1, _) in zip(b, b[1:]):
        assert x0 + nx == x1
    share = [int(work[x0:x0 + nx].sum()) for x0, nx in b]
    assert max(share) <= int(work.sum()) / world + int(work.max())          # within one slab of the ideal
    # degenerate: all the work in one slab still leaves every rank a slab
    w2 = torch.zeros(9, dtype=torch.int64)
    w2[3] = 100
    b2 = slabs.balance_slabs(w2, min(world, 9))
    assert all(nx >= 1 for _, nx in b2) and sum(nx for _, nx in b2) == 9
    with pytest.raises(ValueError):
        slabs.balance_slabs(torch.ones(3), 4)


@pytest.mark.parametrize("cpd,R,world", [(35, 2, 2), (35, 2, 8), (9, 2, 3), (7, 3, 2), (5, 2, 2), (6, 2, 6)])
def test_halo_and_send_plans_are_consistent(cpd, R, world):
    work = torch.ones(cpd)
    b = slabs.balance_slabs(work, world)
    own = slabs.owner_of_slab(b, cpd)
    for r in range(world):
        need = slabs.halo_slabs(b, cpd, R, r)
        x0, nx = b[r]
        mine = {(x0 + i) % cpd for i in range(nx)}
        expect = {(x + d) % cpd for x in mine for d in range(-R, R + 1)} - mine
        assert set(need) == expect and len(need) == len(set(need))
        # what the others send to r is exactly what r needs
        got = []
        for q in range(world):
            got += slabs.send_plan(b, cpd, R, q).get(r, [])
        assert sorted(got) == sorted(need)
        assert all(own[x] != r for x in need)


def test_local_with_ghosts_selects_own_and_halo(oracle_mod):
    cfg = W.scaled(W.CONFIGS[2], 9)
    pos = torch.from_numpy(W.make_positions(cfg))
    b = slabs.balance_slabs(torch.ones(9), 3)
    select, xs = oracle_select(oracle_mod, pos, 9)
    tot = 0
    for r in range(3):
        own, ghost = slabs.local_with_ghosts(select, b, 9, 2, r)
        x0, nx = b[r]
        _, xo = oracle_select(oracle_mod, own, 9)
        assert bool((torch.remainder(xo - x0, 9) < nx).all())
        need = set(slabs.halo_slabs(b, 9, 2, r))
        _, xg = oracle_select(oracle_mod, ghost, 9)
        assert set(xg.tolist()) <= need
        assert ghost.shape[0] == int(sum((xs == x).sum() for x in need))
        tot += own.shape[0]
    assert tot == cfg.N


_WORKER = r'''
import os, sys, json
sys.path.insert(0, os.environ["NF_ROOT"])
import numpy as np, torch
import torch.distributed as dist
import oracle
from paper_2110_11392_b200 import slabs, workloads as W
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
cfg = W.scaled(W.CONFIGS[3], 9)
pos = torch.from_numpy(W.make_positions(cfg))            # every rank generates the same seeded set
def make_select(p):                                      # the oracle's binning stands in for nf_select_slabs on the CPU
    cell, _ = oracle.bin_particles(p.numpy(), cfg.cpd)
    xs = torch.from_numpy(cell // (cfg.cpd * cfg.cpd))
    return lambda x0, nx: p[torch.remainder(xs - x0, cfg.cpd) < nx]
cell, _ = oracle.bin_particles(pos.numpy(), cfg.cpd)
per_slab = np.bincount(cell // (cfg.cpd * cfg.cpd), minlength=cfg.cpd)
bounds = slabs.balance_slabs(per_slab, world)
own, ghost_expect = slabs.local_with_ghosts(make_select(pos), bounds, cfg.cpd, cfg.R, rank)
tail = torch.full((cfg.N, 3), float("nan"))
ghost = slabs.halo_exchange(make_select(own), own, bounds, cfg.cpd, cfg.R, recv_into=lambda n: tail[:n])
key = lambda t: np.sort(np.ascontiguousarray(t.numpy()).view([("x", "f4"), ("y", "f4"), ("z", "f4")]).ravel(), order=["x", "y", "z"])
ok = ghost.shape == ghost_expect.shape and np.array_equal(key(ghost), key(ghost_expect)) and ghost.data_ptr() == tail.data_ptr()
res = torch.tensor([int(ok), own.shape[0], ghost.shape[0]])
out = [torch.zeros_like(res) for _ in range(world)]
dist.all_gather(out, res)
if rank == 0:
    print(json.dumps({"ok": [int(o[0]) for o in out], "own": [int(o[1]) for o in out], "ghost": [int(o[2]) for o in out],
                      "N": cfg.N, "bounds": bounds}))
dist.destroy_process_group()
'''


def test_halo_exchange_two_gloo_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    env = dict(os.environ, NF_ROOT=ROOT)
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29741", str(script)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    r = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert r["ok"] == [1, 1] and sum(r["own"]) == r["N"] and all(g > 0 for g in r["ghost"])
    assert sum(nx for _, nx in r["bounds"]) == 9


# ----------------------------------------------------------------------------- GPU: library-side slab support
@pytest.mark.gpu
def test_cell_histogram_slab_pairs_and_select_match_the_oracle(oracle_mod):
    from paper_2110_11392_b200.binding import NearField
    cfg = W.scaled(W.CONFIGS[3], 9)
    pos_np = W.make_positions(cfg)
    pos_np[:5, 0] = [0.0, np.nextafter(np.float32(1.0), np.float32(0.0)), 1.0 / 9, 2.0 / 9, 0.999999]
    pos_np[5, 0] = 1.25                                    # outside [0, box): wrapped (reading S5)
    pos = torch.from_numpy(pos_np).cuda()
    cell, _ = oracle_mod.bin_particles(pos_np, cfg.cpd)
    offsets, _ = oracle_mod.cell_lists(cell, cfg.cpd)
    n = np.diff(offsets).reshape(cfg.cpd, cfg.cpd, cfg.cpd)
    with NearField(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        counts = nf.cell_histogram(pos)
        assert np.array_equal(counts.cpu().numpy().astype(np.int64), n.ravel())                  # A1's rule, bit exact
        pairs, npart = nf.slab_pairs(counts)
        pairs, npart = pairs.cpu().numpy(), npart.cpu().numpy()
        assert np.array_equal(npart, n.sum(axis=(1, 2)))
        assert int(pairs.sum()) - cfg.N == oracle_mod.pair_count(offsets, cfg.cpd, cfg.R)     # P7, whole box
        x, tot = 4, 0                                                                            # brute force for one slab
        for j in range(cfg.cpd):
            for k in range(cfg.cpd):
                for a in range(-cfg.R, cfg.R + 1):
                    for b in range(-cfg.R, cfg.R + 1):
                        for c in range(-cfg.R, cfg.R + 1):
                            tot += n[x, j, k] * n[(x + a) % cfg.cpd, (j + b) % cfg.cpd, (k + c) % cfg.cpd]
        assert int(pairs[x]) == tot
        xs = cell // (cfg.cpd * cfg.cpd)
        out = torch.empty_like(pos)
        for x0, nx in ((0, 9), (7, 4), (3, 1), (8, 1), (2, 0)):
            k = nf.select_slabs(pos, x0, nx, out=out)
            want = pos_np[((xs - x0) % cfg.cpd) < nx]
            assert k == len(want) == nf.select_slabs(pos, x0, nx)
            assert np.array_equal(out[:k].cpu().numpy(), want)                                 # input order kept
        assert nf.select_slabs(pos[:0], 0, 9) == 0
        bounds = slabs.plan_slabs(nf, pos, 3)
        assert bounds == slabs.balance_slabs(pairs, 3) and sum(nx for _, nx in bounds) == cfg.cpd


@pytest.mark.gpu
def test_histogram_keeps_a_pending_bad_position_flag_and_tiny_selections_work():
    """ nf_cell_histogram used to clear the NaN/Inf flag of an earlier call that nf_sync had not reported
    yet; and nf_select_slabs' block scratch was larger than the N words it borrowed when N <= 3."""
    from paper_2110_11392_b200.binding import NearField, NearFieldError, NF_EPOS
    good = torch.from_numpy(W.uniform(2000, 3)).cuda()
    bad = good.clone()
    bad[17, 1] = float("inf")
    with NearField(7, 2, 1e-3, 1.0) as nf:
        c0 = nf.cell_histogram(good)               # first call on a fresh context: flag starts at zero
        nf.sync()
        assert int(c0.sum()) == 2000
        nf.bin(bad)                                # sets the flag ...
        c1 = nf.cell_histogram(good)               # ... which this call must not clear
        assert int(c1.sum()) == 2000
        with pytest.raises(NearFieldError) as e:
            nf.sync()
        assert e.value.status == NF_EPOS
        c2 = nf.cell_histogram(bad)                # the histogram's own detection: not counted, reported
        with pytest.raises(NearFieldError):
            nf.sync()
        assert int(c2.sum()) == 1999
        nf.bin(good)                               # a new sort starts clean
        nf.sync()
    for n in (1, 2, 3, 4):
        with NearField(7, 2, 1e-3, 1.0) as nf:     # fresh context: scratch sized for exactly n particles
            p = good[:n].contiguous()
            out = torch.empty_like(p)
            assert nf.select_slabs(p, 0, 7, out=out) == n and torch.equal(out, p)
            assert nf.select_slabs(p, 0, 0) == 0


# ----------------------------------------------------------------------------- GPU: emulated decomposition
@pytest.mark.gpu
@pytest.mark.parametrize("label,cfg,world", [("cfg2@13 x3", W.scaled(W.CONFIGS[2], 13), 3),
                                             ("cfg3@10 x4", W.scaled(W.CONFIGS[3], 10), 4),
                                             ("cfg5@9 R3 x2", W.scaled(W.CONFIGS[5], 9), 2),
                                             ("cfg2@5 (=2R+1) x2", W.scaled(W.CONFIGS[2], 5), 2)])
def test_emulated_slab_decomposition_matches_single_call_and_oracle(oracle_mod, label, cfg, world):
    """Ranks run one after the other on one GPU (no kernel waits on another: see the profiling
    guide): each takes its own slabs + ghosts (nf_select_slabs), calls nf_accel with
    nf_set_sink_slabs, and the union must equal the undecomposed result within the parity bar;
    pair counts add up exactly."""
    from paper_2110_11392_b200.binding import NearField
    assert torch.cuda.is_available()
    pos_np = W.make_positions(cfg)
    pos = torch.from_numpy(pos_np).cuda()
    ref, ref_pairs = oracle_mod.accel(pos_np, cfg.cpd, cfg.R, cfg.eps_p)
    cell, _ = oracle_mod.bin_particles(pos_np, cfg.cpd)
    xs = torch.from_numpy(cell // (cfg.cpd * cfg.cpd)).cuda()
    got = torch.full_like(pos, float("nan"))
    pairs = 0
    with NearField(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as planner:
        bounds = slabs.plan_slabs(planner, pos, world)

        def select(x0, nx):
            out = torch.empty_like(pos)
            return out[: planner.select_slabs(pos, x0, nx, out=out)]

        parts = [slabs.local_with_ghosts(select, bounds, cfg.cpd, cfg.R, r) for r in range(world)]
    for r, (own, ghost) in enumerate(parts):
        x0, nx = bounds[r]
        idx = torch.nonzero(torch.remainder(xs - x0, cfg.cpd) < nx).ravel()
        assert own.shape[0] == idx.numel() and torch.equal(own, pos[idx])
        allp = torch.cat([own, ghost]).contiguous()
        with NearField(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
            nf.set_gm(1.0 / cfg.N)                       # the global G*m, not 1/(own + ghost)
            nf.set_sink_slabs(x0, nx)
            acc = torch.full_like(allp, float("nan"))
            nf.accel(allp, acc)
            nf.sync()
            pairs += nf.interaction_count()
            assert bool(torch.isnan(acc[own.shape[0]:]).all())       # ghost rows are left untouched
            got[idx] = acc[: own.shape[0]]
    assert pairs == ref_pairs
    g = got.cpu().numpy().astype(np.float64)
    d = np.linalg.norm(g - ref, axis=1)
    a = np.linalg.norm(ref, axis=1)
    rms = np.sqrt((a ** 2).mean())
    assert np.isfinite(g).all()
    assert d.max() <= 1e-5 * rms, f"{label}: {d.max() / rms:.3e}"
    assert np.median(d[a > 0] / a[a > 0]) <= 2e-6


@pytest.mark.gpu
def test_slab_nearfield_single_rank_equals_plain_call():
    """SlabNearField with one rank (no exchange): same result as nf_accel with the same gm; the
    own+ghost buffer is reused between steps; particles outside the rank's slabs are caught."""
    from paper_2110_11392_b200.binding import NearField
    cfg = W.scaled(W.CONFIGS[2], 9)
    pos = torch.from_numpy(W.make_positions(cfg)).cuda()
    with NearField(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        ref = nf.accel(pos).clone()
        nf.sync()
    snf = slabs.SlabNearField(cfg.cpd, cfg.R, cfg.eps_p, 1.0, [(0, cfg.cpd)], gm=1.0 / cfg.N)
    a1 = snf.accel(pos, validate=True).clone()
    a2 = snf.accel(pos)
    torch.cuda.synchronize()
    assert torch.equal(a1, ref) and torch.equal(a2, ref) and snf.n_ghost == 0
    snf.close()
    half = slabs.SlabNearField(cfg.cpd, cfg.R, cfg.eps_p, 1.0, [(0, 4)], gm=1.0 / cfg.N)
    with pytest.raises(ValueError):
        half.accel(pos, validate=True)
    half.close()


@pytest.mark.gpu
def test_slab_nearfield_on_a_side_stream_is_ordered_with_the_current_stream():
    """accel(stream=side): the internal copy of pos_own runs on the current stream and the force on ``side``.
    The call orders the two itself (it did not), so a caller that keeps working on the current
    stream -- changing pos_own right after the call, reading the result without a sync of ``side`` -- is safe."""
    from paper_2110_11392_b200.binding import NearField
    cfg = W.scaled(W.CONFIGS[2], 21)              # 370 k particles: the copy and the force take long enough to overlap
    pos = torch.from_numpy(W.make_positions(cfg)).cuda()
    with NearField(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        ref = nf.accel(pos).clone()
        nf.sync()
    side = torch.cuda.Stream()
    snf = slabs.SlabNearField(cfg.cpd, cfg.R, cfg.eps_p, 1.0, [(0, cfg.cpd)], gm=1.0 / cfg.N)
    for _ in range(3):
        work = pos.clone()
        a = snf.accel(work, stream=side)
        got = a.clone()                           # current stream, no explicit sync with ``side``
        work.zero_()                              # the caller's buffer is its own again
        assert torch.equal(got, ref)
    snf.close()


@pytest.mark.gpu
def test_sink_slab_setter_rejects_bad_ranges():
    from paper_2110_11392_b200.binding import NearField, NearFieldError
    with NearField(7, 2, 1e-3, 1.0) as nf:
        for x0, nx in ((-1, 3), (7, 1), (0, 0), (0, 8)):
            with pytest.raises(NearFieldError):
                nf.set_sink_slabs(x0, nx)
        nf.set_sink_slabs(6, 7)
