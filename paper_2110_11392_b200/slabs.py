"""Multi-GPU form of the near-field path: 1-D x-slab decomposition with an R-slab halo.

The paper's parallel code decomposes the box into slabs along x ("1-D slab
decomposition", sec. 4.4) and the near field of a slab needs the R slabs on
either side (near-field radius, Table 1).  Here: one process per GPU, each rank
owns a contiguous periodic range of x slabs balanced by PAIR COUNT (not slab count), receives
the particles of the R ghost slabs on each side from their owners (one point-to-point exchange,
``torch.distributed`` isend/irecv: NCCL between GPUs, gloo in the CPU tests) straight into the
tail of its own+ghost buffer, and calls ``nf_accel`` with ``nf_set_sink_slabs`` so that only its
own slabs are sinks.  Every sink is owned by exactly one rank, so there is no reduction.

Everything here is host-side plumbing: slab index arithmetic, message sizes, send/recv.  The
method's arithmetic stays in the CUDA library: which cell a particle is in (``nf_cell_histogram``,
``nf_select_slabs`` -- step A1's rule), the pair count per slab (``nf_slab_pairs`` -- identity P7)
and the forces.  The functions that need particles take a ``select(x0, nx) -> tensor`` callable for
that reason: ``SlabNearField`` passes the library's; the CPU tests of the plumbing pass their own.
"""
from __future__ import annotations

from typing import Callable

import torch


# ----------------------------------------------------------------------------- planning (integers only)
def balance_slabs(work, world: int) -> list[tuple[int, int]]:
    """Cut the cpd slabs into ``world`` contiguous ranges [(x0, nx)] of nearly equal work, each
    with at least one slab (cut k goes where the prefix sum first reaches k/world of the total).
    ``work``: per-slab work (``nf_slab_pairs``), any sequence or 1-D tensor of integers."""
    w = [int(v) for v in (work.tolist() if hasattr(work, "tolist") else work)]
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


def slab_runs(slabs: list[int], cpd: int) -> list[tuple[int, int]]:
    """a set of slab indices as periodic runs [(x0, nx)] (a halo is one or two of them)"""
    left = sorted(set(slabs))
    runs: list[tuple[int, int]] = []
    while left:
        s = set(left)
        x0 = next((x for x in left if (x - 1) % cpd not in s), left[0])     # a run start (any slab if the set is a full circle)
        n = 1
        while (x0 + n) % cpd in s and n < len(s):
            n += 1
        runs.append((x0, n))
        gone = {(x0 + i) % cpd for i in range(n)}
        left = [x for x in left if x not in gone]
    return runs


# ----------------------------------------------------------------------------- exchange
Select = Callable[[int, int], torch.Tensor]     # (x0, nx) -> the local particles in x slabs [x0, x0+nx), [n,3]


def halo_exchange(select: Select, like: torch.Tensor, bounds: list[tuple[int, int]], cpd: int, R: int, group=None,
                  recv_into: Callable[[int], torch.Tensor] | None = None) -> torch.Tensor:
    """Send the particles of my boundary slabs to the ranks that need them and receive my ghosts.
    One count exchange (all_gather of a [world] vector) and one batch of isend/irecv.
    ``like``: any tensor of the particles' dtype/device.  ``recv_into(n)``: a contiguous [n,3] view
    to receive the n ghosts into (the tail of the caller's own+ghost buffer); default: a new tensor.
    Returns that view."""
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return like.new_zeros((0, 3))
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    out = {}
    counts = torch.zeros(world, dtype=torch.int64, device=like.device)
    for q, need in send_plan(bounds, cpd, R, rank).items():
        parts = [select(x0, nx) for x0, nx in slab_runs(need, cpd)]
        out[q] = parts[0] if len(parts) == 1 else torch.cat(parts, dim=0)
        counts[q] = out[q].shape[0]
    allc = [torch.zeros_like(counts) for _ in range(world)]
    dist.all_gather(allc, counts, group=group)
    nrecv = {q: int(allc[q][rank]) for q in range(world) if q != rank}
    total = sum(nrecv.values())
    ghosts = recv_into(total) if recv_into is not None else like.new_empty((total, 3))
    peer = (lambda q: dist.get_global_rank(group, q)) if group is not None else (lambda q: q)
    ops, at = [], 0
    for q in sorted(nrecv):
        if nrecv[q]:
            ops.append(dist.P2POp(dist.irecv, ghosts[at:at + nrecv[q]], peer(q), group))
            at += nrecv[q]
        if q in out and out[q].shape[0]:
            ops.append(dist.P2POp(dist.isend, out[q], peer(q), group))
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    return ghosts


def local_with_ghosts(select: Select, bounds: list[tuple[int, int]], cpd: int, R: int, rank: int):
    """No-communication form for a process that can see every particle (tests, single-GPU emulation
    of a decomposition): -> (pos_own, pos_ghost) of ``rank`` from a ``select`` over ALL particles."""
    x0, nx = bounds[rank]
    own = select(x0, nx)
    runs = slab_runs(halo_slabs(bounds, cpd, R, rank), cpd)
    parts = [select(a, n) for a, n in runs]
    ghost = torch.cat(parts, dim=0) if parts else own.new_zeros((0, 3))
    return own, ghost


# ----------------------------------------------------------------------------- the sharded call
def plan_slabs(nf, pos_own: torch.Tensor, world: int, group=None) -> list[tuple[int, int]]:
    """pair-balanced slab ranges from the ranks' particles: local histogram (``nf_cell_histogram``),
    one all_reduce of cpd^3 int32, pairs per slab (``nf_slab_pairs``), cuts on the host."""
    import torch.distributed as dist
    counts = nf.cell_histogram(pos_own)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(counts, group=group)
    pairs, _ = nf.slab_pairs(counts)
    return balance_slabs(pairs.cpu(), world)


class SlabNearField:
    """nf_accel over a slab decomposition: ``accel(pos_own)`` -> accelerations of the rank's own
    particles.  ``bounds`` = [(x0, nx)] per rank (``plan_slabs`` / ``balance_slabs``); every particle
    of ``pos_own`` must lie in the rank's slabs (``validate=True`` checks it on the device).
    ``gm`` = G*m of the WHOLE particle set (1/N_global for the paper's unit total mass): the default
    of the single-GPU call, 1/N of the call, would be 1/(own + ghost) here and differ between ranks."""

    def __init__(self, cpd: int, R: int, eps_plummer: float, box: float, bounds, gm: float, group=None):
        import torch.distributed as dist
        from .binding import NearField
        self.cpd, self.R, self.box, self.bounds, self.group = cpd, R, box, list(bounds), group
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.nf = NearField(cpd, R, eps_plummer, box)
        self.nf.set_gm(gm)
        x0, nx = self.bounds[self.rank]
        self.nf.set_sink_slabs(x0, nx)
        self.n_ghost = 0
        self.halo_bytes = 0          # bytes received in the last exchange
        self._buf = self._acc = self._send = None

    def _room(self, like: torch.Tensor, n: int):
        if self._buf is None or self._buf.shape[0] < n:
            cap = int(n * 1.05) + 1024
            old = self._buf
            self._buf = like.new_empty((cap, 3))
            self._acc = like.new_zeros((cap, 3))
            if old is not None:
                self._buf[: old.shape[0]] = old

    def accel(self, pos_own: torch.Tensor, stream=None, validate: bool = False) -> torch.Tensor:
        n_own = pos_own.shape[0]
        x0, nx = self.bounds[self.rank]
        if validate and self.nf.select_slabs(pos_own, x0, nx) != n_own:
            raise ValueError("pos_own holds particles outside this rank's slabs")
        if self._send is None or self._send.shape[0] < n_own:
            self._send = pos_own.new_empty((n_own, 3))
        self._room(pos_own, n_own + max(self.n_ghost, n_own // 8))
        self._buf[:n_own].copy_(pos_own)

        def select(a, n):
            k = self.nf.select_slabs(pos_own, a, n, out=self._send)
            return self._send[:k].clone()

        def recv_into(n):
            self._room(pos_own, n_own + n)
            return self._buf[n_own:n_own + n]

        ghosts = halo_exchange(select, pos_own, self.bounds, self.cpd, self.R, self.group, recv_into)
        self.n_ghost = int(ghosts.shape[0])
        self.halo_bytes = self.n_ghost * 12
        n_tot = n_own + self.n_ghost
        # The copy into _buf, the slab selection and the halo receive ran on torch's CURRENT stream; the force call
        # runs on ``stream``.  When the two differ they are ordered here in both directions: the force waits for
        # own + ghost rows to be complete, and the current stream waits for the force, so that the returned view (and
        # the next call's writes into _buf / _acc) are safe for a caller that keeps working on the current stream.
        cur = torch.cuda.current_stream(pos_own.device) if pos_own.is_cuda else None
        if stream is not None and cur is not None and stream != cur:
            stream.wait_stream(cur)
        self.nf.accel(self._buf[:n_tot], self._acc[:n_tot], stream=stream)      # ghost rows of acc are not written
        if stream is not None and cur is not None and stream != cur:
            cur.wait_stream(stream)
        return self._acc[:n_own]

    def interaction_count(self) -> int:
        return self.nf.interaction_count()

    def close(self):
        self.nf.close()
