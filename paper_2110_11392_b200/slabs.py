"""Multi-GPU form of the near-field path: 1-D x-slab decomposition with an R-slab halo.

The paper's parallel code decomposes the box into slabs along x ("1-D slab
decomposition", sec. 4.4) and the near field of a slab needs the R slabs on
either side (near-field radius, Table 1).  Here: one process per GPU, each rank
owns a contiguous periodic range of x slabs balanced by PAIR COUNT (not slab count), receives
the particles of the R ghost slabs on each side from their owners (one point-to-point exchange,
``torch.distributed`` isend/irecv: NCCL between GPUs, gloo in the CPU tests), and calls
``nf_accel`` with ``nf_set_sink_slabs`` so that only its own slabs are sinks.  Every sink is owned
by exactly one rank, so there is no reduction.

Everything here is host-side plumbing (index arithmetic, message sizes, send/recv); the force
arithmetic stays in the CUDA library.  ``slab_index`` repeats the library's cell rule
(reading S5: floor((double)x * CPD / box) mod CPD) because the owner of a particle
must be known before it is sent.
"""
from __future__ import annotations

import torch


# ----------------------------------------------------------------------------- planning
def slab_index(pos: torch.Tensor, cpd: int, box: float = 1.0) -> torch.Tensor:
    """x cell index of every particle (int64, same device): floor((double)x * CPD / box) mod CPD."""
    t = pos[:, 0].to(torch.float64) * (float(cpd) / float(box))
    return torch.remainder(torch.floor(t).to(torch.int64), cpd)


def cell_index(pos: torch.Tensor, cpd: int, box: float = 1.0) -> torch.Tensor:
    t = torch.floor(pos.to(torch.float64) * (float(cpd) / float(box))).to(torch.int64)
    c = torch.remainder(t, cpd)
    return (c[:, 0] * cpd + c[:, 1]) * cpd + c[:, 2]


def pairs_per_slab(counts: torch.Tensor, cpd: int, R: int) -> torch.Tensor:
    """counts: occupancy histogram [cpd^3] (key = (cx*cpd+cy)*cpd+cz).  Returns, per x slab, the
    number of (sink, source) pairs whose sink lies in the slab: sum_c n_c (B*n)_c with B the
    periodic (2R+1)^3 box filter (the integer identity P7 of DESIGN.md), int64 [cpd]."""
    n = counts.to(torch.int64).reshape(cpd, cpd, cpd)
    f = n
    for dim in range(3):
        acc = torch.zeros_like(f)
        for s in range(-R, R + 1):
            acc += torch.roll(f, shifts=s, dims=dim)
        f = acc
    return (n * f).sum(dim=(1, 2))


def balance_slabs(work: torch.Tensor, world: int) -> list[tuple[int, int]]:
    """Cut the cpd slabs into ``world`` contiguous ranges [(x0, nx)] of nearly equal work, each
    with at least one slab (cut k goes where the prefix sum first reaches k/world of the total)."""
    w = [int(v) for v in work.tolist()]
    cpd = len(w)
    if world > cpd:
        raise ValueError(f"{world} ranks need at least {world} slabs, the grid has {cpd}")
    prefix = [0]
    for v in w:
        prefix.append(prefix[-1] + v)          # prefix[x] = work of slabs 0 .. x-1
    total = prefix[-1]
    cuts = [0]
    for k in range(1, world):
        lo, hi = cuts[-1] + 1, cpd - (world - k)     # leave one slab for every rank
        x = lo
        while x < hi and prefix[x] * world < k * total:
            x += 1
        cuts.append(x)
    cuts.append(cpd)
    return [(cuts[i], cuts[i + 1] - cuts[i]) for i in range(world)]


def owner_of_slab(bounds: list[tuple[int, int]], cpd: int) -> list[int]:
    own = [-1] * cpd
    for r, (x0, nx) in enumerate(bounds):
        for x in range(x0, x0 + nx):
            own[x % cpd] = r
    assert all(o >= 0 for o in own), "slab ranges do not cover the grid"
    return own


def halo_slabs(bounds: list[tuple[int, int]], cpd: int, R: int, rank: int) -> list[int]:
    """the ghost slabs ``rank`` needs: within R slabs of its range (periodic), not its own, each once."""
    x0, nx = bounds[rank]
    mine = {x % cpd for x in range(x0, x0 + nx)}
    need = []
    for x in list(range(x0 - R, x0)) + list(range(x0 + nx, x0 + nx + R)):
        xm = x % cpd
        if xm not in mine and xm not in need:
            need.append(xm)
    return need


def send_plan(bounds: list[tuple[int, int]], cpd: int, R: int, rank: int) -> dict[int, list[int]]:
    """{destination rank: the slabs of ``rank`` it must send there}"""
    own = owner_of_slab(bounds, cpd)
    plan: dict[int, list[int]] = {}
    for q in range(len(bounds)):
        if q == rank:
            continue
        s = [x for x in halo_slabs(bounds, cpd, R, q) if own[x] == rank]
        if s:
            plan[q] = s
    return plan


# ----------------------------------------------------------------------------- exchange
def halo_exchange(pos_own: torch.Tensor, xslab_own: torch.Tensor, bounds: list[tuple[int, int]], cpd: int, R: int,
                  group=None) -> torch.Tensor:
    """Send the particles of my boundary slabs to the ranks that need them and return the ghost
    particles I receive ([n_ghost, 3], same dtype/device as pos_own).  One count exchange
    (all_gather of a [world] vector) and one batch of isend/irecv."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    if world == 1:
        return pos_own.new_zeros((0, 3))
    plan = send_plan(bounds, cpd, R, rank)
    out = {}
    counts = torch.zeros(world, dtype=torch.int64, device=pos_own.device)
    for q, slabs in plan.items():
        m = torch.zeros(cpd, dtype=torch.bool, device=pos_own.device)
        m[torch.tensor(slabs, device=pos_own.device)] = True
        out[q] = pos_own[m[xslab_own]].contiguous()
        counts[q] = out[q].shape[0]
    allc = [torch.zeros_like(counts) for _ in range(world)]
    dist.all_gather(allc, counts, group=group)
    ops, recv = [], {}
    for q in range(world):
        if q == rank:
            continue
        nrecv = int(allc[q][rank])
        if nrecv:
            recv[q] = pos_own.new_empty((nrecv, 3))
            ops.append(dist.P2POp(dist.irecv, recv[q], dist.get_global_rank(group, q) if group is not None else q, group))
        if q in out and out[q].shape[0]:
            ops.append(dist.P2POp(dist.isend, out[q], dist.get_global_rank(group, q) if group is not None else q, group))
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    if not recv:
        return pos_own.new_zeros((0, 3))
    return torch.cat([recv[q] for q in sorted(recv)], dim=0)


def local_with_ghosts(pos_all: torch.Tensor, bounds: list[tuple[int, int]], cpd: int, R: int, rank: int, box: float = 1.0):
    """No-communication form for a rank that can see every particle (tests, single-GPU emulation
    of a decomposition): -> (pos_own, pos_ghost) of ``rank``."""
    xs = slab_index(pos_all, cpd, box)
    x0, nx = bounds[rank]
    own = torch.remainder(xs - x0, cpd) < nx
    ghost_slabs = halo_slabs(bounds, cpd, R, rank)
    g = torch.zeros(cpd, dtype=torch.bool, device=pos_all.device)
    if ghost_slabs:
        g[torch.tensor(ghost_slabs, device=pos_all.device)] = True
    return pos_all[own], pos_all[g[xs] & ~own]


# ----------------------------------------------------------------------------- the sharded call
class SlabNearField:
    """nf_accel over a slab decomposition: ``accel(pos_own)`` -> accelerations of the rank's own
    particles.  ``bounds`` = [(x0, nx)] per rank (``balance_slabs``); every particle of
    ``pos_own`` must lie in the rank's slabs."""

    def __init__(self, cpd: int, R: int, eps_plummer: float, box: float, bounds, group=None):
        import torch.distributed as dist
        from .binding import NearField
        self.cpd, self.R, self.box, self.bounds, self.group = cpd, R, box, list(bounds), group
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.nf = NearField(cpd, R, eps_plummer, box)
        x0, nx = self.bounds[self.rank]
        self.nf.set_sink_slabs(x0, nx)
        self.n_ghost = 0

    def accel(self, pos_own: torch.Tensor, stream=None) -> torch.Tensor:
        xs = slab_index(pos_own, self.cpd, self.box)
        x0, nx = self.bounds[self.rank]
        if not bool((torch.remainder(xs - x0, self.cpd) < nx).all()):
            raise ValueError("pos_own holds particles outside this rank's slabs")
        ghosts = halo_exchange(pos_own, xs, self.bounds, self.cpd, self.R, self.group)
        self.n_ghost = int(ghosts.shape[0])
        allp = torch.cat([pos_own, ghosts], dim=0).contiguous()
        acc = torch.zeros_like(allp)
        self.nf.accel(allp, acc, stream=stream)
        return acc[: pos_own.shape[0]]

    def interaction_count(self) -> int:
        return self.nf.interaction_count()

    def close(self):
        self.nf.close()
