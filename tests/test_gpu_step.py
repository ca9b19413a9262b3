"""nf_kick_drift and nf_timestep_ratio (Table 1 :379-380) against the oracle.
Kick/Drift: bit-exact (both sides evaluate each update in double with separately rounded product
and sum, and round to float32 once).  Time-step ratio: double sums in a different order: 1e-12."""
import numpy as np
import pytest

from paper_2110_11392_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    return torch


@pytest.fixture(scope="module")
def NF():
    from paper_2110_11392_b200.binding import NearField
    return NearField


def _state(cfg, seed):
    rng = np.random.default_rng(seed)
    pos = W.make_positions(cfg)
    vel = (rng.normal(size=pos.shape) * 0.3).astype(np.float32)
    acc = (rng.normal(size=pos.shape) * 5.0).astype(np.float32)
    return pos, vel, acc


@pytest.mark.parametrize("label,cfg", [("cfg1", W.CONFIGS[1]), ("cfg3 @cpd10", W.scaled(W.CONFIGS[3], 10)), ("cfg2 full", W.CONFIGS[2])])
@pytest.mark.parametrize("dtk,dtd", [(0.01, 0.02), (0.005, 0.0), (0.0, 0.7), (-0.01, -0.02)])
def test_kick_drift_bit_exact(torch_cuda, NF, oracle_mod, label, cfg, dtk, dtd):
    pos, vel, acc = _state(cfg, 1)
    rp, rv = oracle_mod.kick_drift(pos, vel, acc, dtk, dtd)
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        dp, dv, da = (torch_cuda.from_numpy(x.copy()).cuda() for x in (pos, vel, acc))
        nf.kick_drift(dp, dv, da, dtk, dtd)
        torch_cuda.cuda.synchronize()
        gp, gv = dp.cpu().numpy(), dv.cpu().numpy()
    assert np.array_equal(gv, rv)
    assert np.array_equal(gp, rp)
    assert np.all((gp >= 0) & (gp < 1))


def test_kick_drift_other_box_and_empty(torch_cuda, NF, oracle_mod):
    rng = np.random.default_rng(2)
    pos = (rng.random((5000, 3)) * 5).astype(np.float32)
    vel = rng.normal(size=pos.shape).astype(np.float32) * 3
    acc = rng.normal(size=pos.shape).astype(np.float32)
    rp, rv = oracle_mod.kick_drift(pos, vel, acc, 0.1, 2.0, box=5.0)
    with NF(7, 2, 1e-3, 5.0) as nf:
        dp, dv, da = (torch_cuda.from_numpy(x.copy()).cuda() for x in (pos, vel, acc))
        nf.kick_drift(dp, dv, da, 0.1, 2.0)
        e = torch_cuda.zeros((0, 3), dtype=torch_cuda.float32, device="cuda")
        nf.kick_drift(e, e, e, 0.1, 0.1)
        torch_cuda.cuda.synchronize()
        assert np.array_equal(dp.cpu().numpy(), rp) and np.array_equal(dv.cpu().numpy(), rv)
        assert float(dp.max()) < 5.0 and float(dp.min()) >= 0.0


@pytest.mark.parametrize("label,cfg", [("cfg1", W.CONFIGS[1]), ("cfg3 @cpd10", W.scaled(W.CONFIGS[3], 10)), ("cfg5 @cpd9", W.scaled(W.CONFIGS[5], 9))])
def test_timestep_ratio(torch_cuda, NF, oracle_mod, label, cfg):
    pos, vel, acc = _state(cfg, 3)
    cell, _ = oracle_mod.bin_particles(pos, cfg.cpd)
    acc[cell == cell[0]] = 0                              # one cell without acceleration: must not constrain
    ref = oracle_mod.timestep_ratio(pos, vel, acc, cfg.cpd)
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        got = nf.timestep_ratio(*(torch_cuda.from_numpy(x).cuda() for x in (pos, vel, acc)))
        none = nf.timestep_ratio(torch_cuda.from_numpy(pos).cuda(), torch_cuda.from_numpy(vel).cuda(),
                                 torch_cuda.zeros_like(torch_cuda.from_numpy(acc)).cuda())
    assert np.allclose(got, ref, rtol=1e-12, atol=0), (got, ref)
    assert got[3] == ref[3]                               # a maximum: exact
    assert np.isinf(none[0]) and np.isinf(none[1]) and none[3] == 0.0


def test_leapfrog_step_with_the_near_field(torch_cuda, NF, oracle_mod):
    """one KDK step driven by nf_accel on the GPU against the same step driven by the oracle's
    accelerations: positions agree to float32 rounding of a 1e-5-accurate acceleration."""
    cfg = W.scaled(W.CONFIGS[2], 9)
    pos = W.make_positions(cfg)
    vel = np.zeros_like(pos)
    dt = 1e-3
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        dp, dv = torch_cuda.from_numpy(pos.copy()).cuda(), torch_cuda.from_numpy(vel.copy()).cuda()
        a0 = nf.accel(dp)
        nf.kick_drift(dp, dv, a0, dt / 2, dt)
        a1 = nf.accel(dp)
        nf.kick_drift(dp, dv, a1, dt / 2, 0.0)
        nf.sync()
        gp, gv = dp.cpu().numpy(), dv.cpu().numpy()
    r0, _ = oracle_mod.accel(pos, cfg.cpd, cfg.R, cfg.eps_p)
    p1, v1 = oracle_mod.kick_drift(pos, vel, r0.astype(np.float32), dt / 2, dt)
    r1, _ = oracle_mod.accel(p1, cfg.cpd, cfg.R, cfg.eps_p)
    _, v2 = oracle_mod.kick_drift(p1, v1, r1.astype(np.float32), dt / 2, 0.0)
    d = np.abs(gp.astype(np.float64) - p1)
    d = np.minimum(d, 1 - d)
    assert d.max() <= 2e-7
    vr = np.sqrt((v2.astype(np.float64) ** 2).sum(1).mean())
    assert np.abs(gv - v2).max() <= 2e-5 * vr


def test_bin_once_reuse_everywhere(torch_cuda, NF, oracle_mod):
    """nf_bin pins the grid order of a position buffer: the force, f64, multipole, Taylor and
    time-step calls of one step then reuse it (no re-sort: fewer launches, stage times of A1-A3
    read 0) with bit-identical results; moving the particles (nf_kick_drift) or passing another
    buffer drops the pin."""
    torch = torch_cuda
    cfg = W.scaled(W.CONFIGS[3], 10)
    pos, vel, acc_in = _state(cfg, 5)
    d_pos, d_vel = torch.from_numpy(pos).cuda(), torch.from_numpy(vel).cuda()
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        nf.set_option("stage_timing", 1)
        n0 = nf.launch_count()
        a_plain = nf.accel(d_pos).clone()
        plain_launches = nf.launch_count() - n0
        M_plain = nf.multipoles(d_pos, 4).clone()
        f_plain = nf.accel_f64(d_pos).clone()
        t_plain = nf.timestep_ratio(d_pos, d_vel, a_plain)
        nf.bin(d_pos)
        n1 = nf.launch_count()
        a_pin = nf.accel(d_pos).clone()
        pinned_launches = nf.launch_count() - n1
        st = nf.stage_ms()
        assert pinned_launches <= plain_launches - 6          # key_hist, 3 scans, scatter, rank_gather not launched
        assert st["A1_key_hist"] < 0.02 and st["A3_scatter_rank_gather"] < 0.02 and st["A5_interact_A6_unpermute"] > 0   # back-to-back events
        n2 = nf.launch_count()
        M_pin = nf.multipoles(d_pos, 4)
        assert nf.launch_count() - n2 == 1
        f_pin = nf.accel_f64(d_pos)
        torch.manual_seed(1)
        T = torch.randn_like(M_pin)
        y_pin = nf.taylor_accel(d_pos, T, 4).clone()
        t_pin = nf.timestep_ratio(d_pos, d_vel, a_plain)
        dbg = nf.debug_cells()
        nf.sync()
        assert torch.equal(a_pin, a_plain) and torch.equal(M_pin, M_plain) and torch.equal(f_pin, f_plain)
        assert np.allclose(t_pin, t_plain, rtol=1e-13, atol=0)      # (a double sum by atomics: order varies)
        cell, _ = oracle_mod.bin_particles(pos, cfg.cpd)
        offsets, order = oracle_mod.cell_lists(cell, cfg.cpd)
        assert np.array_equal(dbg["offsets"].astype(np.int64), offsets) and np.array_equal(dbg["perm"].astype(np.int64), order)
        # another buffer: sorted as usual, and the pin is gone
        other = torch.from_numpy(W.uniform(3000, 9)).cuda()
        b0 = nf.accel(other).clone()
        n3 = nf.launch_count()
        nf.accel(d_pos)
        assert nf.launch_count() - n3 == plain_launches
        # pinned again, then the particles move: the next call sorts the new positions
        nf.bin(d_pos)
        nf.kick_drift(d_pos, d_vel, a_plain, 0.0, 0.05)
        a_moved = nf.accel(d_pos)
        y_unpinned = nf.taylor_accel(torch.from_numpy(pos).cuda(), T, 4)
        nf.sync()
        moved = d_pos.cpu().numpy()
        assert torch.equal(y_unpinned, y_pin)
    ref, _ = oracle_mod.accel(moved, cfg.cpd, cfg.R, cfg.eps_p)
    g = a_moved.cpu().numpy().astype(np.float64)
    rms = np.sqrt((ref ** 2).sum(1).mean())
    assert np.linalg.norm(g - ref, axis=1).max() <= 1e-5 * rms
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf2:
        assert torch.equal(nf2.accel(other), b0)


REBIN = [("cfg2 @cpd13", W.scaled(W.CONFIGS[2], 13)), ("cfg3 @cpd10", W.scaled(W.CONFIGS[3], 10)), ("cfg4 @cpd9", W.scaled(W.CONFIGS[4], 9)),
         ("cfg5 @cpd7 R3", W.scaled(W.CONFIGS[5], 7)), ("cfg3 full", W.CONFIGS[3])]


@pytest.mark.parametrize("label,cfg", REBIN, ids=[r[0] for r in REBIN])
def test_rebin_equals_a_full_sort(torch_cuda, NF, oracle_mod, label, cfg):
    """nf_rebin (insert list + merge) after the particles moved: cell offsets, the
    permutation (ascending input index within a cell), the cell-relative planes and the padding equal
    a full counting sort of the new positions bit for bit -- for drifts that move a few per cent of the
    particles out of their cells, about half of them, and all of them, several steps in a row."""
    torch = torch_cuda
    pos, vel, _ = _state(cfg, 7)
    vel = (vel / 0.3 * cfg.cell).astype(np.float32)               # rms 1 cell per unit time per component
    d_pos, d_vel = torch.from_numpy(pos.copy()).cuda(), torch.from_numpy(vel).cuda()
    zero = torch.zeros_like(d_pos)
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf, NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as fresh:
        nf.bin(d_pos)
        for step, dt in enumerate((0.02, 0.0, 0.4, 5.0, 0.05)):
            before = d_pos.clone()
            nf.kick_drift(d_pos, d_vel, zero, 0.0, dt)
            nf.rebin(d_pos)
            got = nf.debug_cells()
            moved = d_pos.cpu().numpy()
            cell, _ = oracle_mod.bin_particles(moved, cfg.cpd)
            offsets, order = oracle_mod.cell_lists(cell, cfg.cpd)
            assert np.array_equal(got["offsets"].astype(np.int64), offsets), (label, step)
            assert np.array_equal(got["perm"].astype(np.int64), order), (label, step)
            fresh.bin(d_pos)
            ref = fresh.debug_cells()
            for k in ("offsets", "perm", "poffsets", "sorted_key"):
                assert np.array_equal(got[k], ref[k]), (label, step, k)
            assert np.array_equal(got["sorted_xyz"], ref["sorted_xyz"]), (label, step)
            if cfg.N < 2_000_000:
                a = nf.accel(d_pos)                                 # on the updated order (pinned by nf_rebin)
                b = fresh.accel(d_pos)
                nf.sync(), fresh.sync()
                assert torch.equal(a, b), (label, step)
            old_cell, _ = oracle_mod.bin_particles(before.cpu().numpy(), cfg.cpd)
            frac = float((old_cell != cell).mean())
            assert (dt == 0.0) == (frac == 0.0)
        assert frac < 0.2                                           # the last drift is a small one again


def test_rebin_without_a_binning_and_with_another_count(torch_cuda, NF, oracle_mod):
    torch = torch_cuda
    cfg = W.scaled(W.CONFIGS[2], 9)
    pos = W.make_positions(cfg)
    d = torch.from_numpy(pos).cuda()
    with NF(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        nf.rebin(d)                                                 # nothing held yet: a full sort
        cell, _ = oracle_mod.bin_particles(pos, cfg.cpd)
        offsets, order = oracle_mod.cell_lists(cell, cfg.cpd)
        g = nf.debug_cells()
        assert np.array_equal(g["offsets"].astype(np.int64), offsets) and np.array_equal(g["perm"].astype(np.int64), order)
        half = d[: cfg.N // 2].contiguous()
        nf.rebin(half)                                              # another count: a full sort again
        c2, _ = oracle_mod.bin_particles(pos[: cfg.N // 2], cfg.cpd)
        o2, r2 = oracle_mod.cell_lists(c2, cfg.cpd)
        g = nf.debug_cells()
        assert np.array_equal(g["offsets"].astype(np.int64), o2) and np.array_equal(g["perm"].astype(np.int64), r2)
        # everything into one cell, then spread out again
        gen = torch.Generator(device="cuda").manual_seed(5)        # seeded, and away from the cell's upper face: (3 + u)/cpd must not round into cell 4
        one = ((3 + 0.999 * torch.rand((cfg.N // 2, 3), device="cuda", generator=gen)) / cfg.cpd).contiguous()
        nf.rebin(one)
        g = nf.debug_cells()
        assert int(g["offsets"][-1]) == cfg.N // 2 and int(np.diff(g["offsets"].astype(np.int64)).max()) == cfg.N // 2
        assert np.array_equal(g["perm"], np.arange(cfg.N // 2, dtype=np.uint32))
        nf.rebin(half)
        g = nf.debug_cells()
        assert np.array_equal(g["offsets"].astype(np.int64), o2) and np.array_equal(g["perm"].astype(np.int64), r2)


def test_long_cells_in_every_rank_regime(torch_cuda, NF, oracle_mod):
    """A3's stable order (ascending input index within a cell) for cells of every size class of the
    binner: up to one 256-slot chunk (rank by counting), up to 8192 and up to 32768 (bitonic sort in
    shared memory, two launches), beyond that (sorted chunks + binary searches) -- input order shuffled,
    bit-exact against the oracle's counting sort; then the same through nf_rebin after a small drift."""
    torch = torch_cuda
    rng = np.random.default_rng(21)
    cpd = 5
    sizes = {(0, 0, 0): 40000, (1, 2, 3): 33000, (2, 2, 2): 20000, (3, 1, 0): 8192, (4, 4, 4): 8193, (0, 3, 1): 3000, (2, 0, 4): 257,
             (1, 1, 1): 256, (3, 3, 3): 100, (4, 0, 2): 1}
    parts = [((np.array(c) + rng.random((n, 3))) / cpd) for c, n in sizes.items()]
    pos = np.concatenate(parts)
    pos = pos[rng.permutation(len(pos))].astype(np.float32)
    pos[pos >= 1.0] = 0.0
    d = torch.from_numpy(pos).cuda()
    with NF(cpd, 2, 0.002, 1.0) as nf:
        nf.bin(d)
        cell, off = oracle_mod.bin_particles(pos, cpd)
        offsets, order = oracle_mod.cell_lists(cell, cpd)
        g = nf.debug_cells()
        assert np.array_equal(g["offsets"].astype(np.int64), offsets)
        assert np.array_equal(g["perm"].astype(np.int64), order)
        real = (g["sorted_key"] & 0x80000000) == 0
        assert np.array_equal(g["sorted_key"][real].astype(np.int64), cell[order])
        assert np.all(np.abs(g["sorted_xyz"][real] - off[order] * cpd) <= 1e-6)
        moved = pos.copy()
        moved[::7] = np.mod(moved[::7].astype(np.float64) + 0.03, 1.0).astype(np.float32)
        moved[moved >= 1.0] = 0.0
        d.copy_(torch.from_numpy(moved))
        nf.rebin(d)
        c2, _ = oracle_mod.bin_particles(moved, cpd)
        o2, r2 = oracle_mod.cell_lists(c2, cpd)
        g = nf.debug_cells()
        assert np.array_equal(g["offsets"].astype(np.int64), o2) and np.array_equal(g["perm"].astype(np.int64), r2)
