"""Slab space decomposition over ranks ("space-decomposition"): one process per GPU, each
running the unchanged single-GPU library (cells, Verlet lists, VERTEX / EDGE forces) on the particles it owns plus ghost
copies of its two neighbours' particles within the halo width r_v = rcut + skin of its slab.

What runs where
  * every arithmetic step on particle data is a kernel of libmd_b200.so: md_half_step (kick / drift / skin check),
    md_dd_select (which particles leave the slab, which sit in a halo zone), md_gather_ids / md_scatter_ids (pack / unpack),
    md_build_* and md_forces;
  * this module owns the PROTOCOL (who sends what to whom, when the ranks rebuild) and moves bytes: torch.distributed
    point-to-point (NCCL over NVLink between GPUs, gloo in the CPU tests), or an in-process transport when several
    domains live in one process (single-GPU tests of the protocol; nothing is timed there).

One step:   kick+drift -> forward halo (positions, quaternions of the send lists) -> all-reduce(max) of the skin flags
            -> [rebuild: wrap, migration, new halo, md_resize, md_bind_state, cells, lists] -> forces -> kick.
Pairs across a slab face are evaluated by both ranks (each sees the other's particle as a ghost): redundant arithmetic
instead of a reverse force exchange, so EDGE needs no force halo either.  Ghost forces are discarded.  NVE only.
"""
from __future__ import annotations

import ctypes as C
from typing import List, Optional

import numpy as np

from .binding import ARRAY, MDSystem


# ------------------------------------------------------------------------------------------------
# host logic: the slab plan (no GPU needed; tests/test_dd_gloo.py)
# ------------------------------------------------------------------------------------------------
class SlabPlan:
    """P slabs along x.  Bounds are fp32 values (coordinates are fp32): slab k = [b[k], b[k+1]), b[P] = Lx."""

    def __init__(self, box, nranks: int, halo: float):
        self.box = np.ascontiguousarray(box, dtype=np.float64)
        self.nranks = int(nranks)
        self.halo = float(halo)
        Lx = float(self.box[0])
        b = [np.float32(k * Lx / self.nranks) for k in range(self.nranks)] + [np.float32(Lx)]
        self.bounds = np.array(b, dtype=np.float32)
        width = float(np.min(np.diff(self.bounds.astype(np.float64))))
        if self.nranks > 1 and width < 2.0 * self.halo:
            raise ValueError(f"slab width {width:.3f} < 2 x halo {self.halo:.3f}: too many ranks for this box")

    def slab(self, rank: int):
        return float(self.bounds[rank]), float(self.bounds[rank + 1])

    def left(self, rank: int) -> int:
        return (rank - 1) % self.nranks

    def right(self, rank: int) -> int:
        return (rank + 1) % self.nranks

    def zone_to_left(self, rank: int):
        """Owned particles the LEFT neighbour needs as ghosts: within `halo` of this slab's lower face."""
        lo, _ = self.slab(rank)
        return lo, float(np.float32(lo + self.halo))

    def zone_to_right(self, rank: int):
        _, hi = self.slab(rank)
        return float(np.float32(hi - self.halo)), hi

    def owner(self, x) -> np.ndarray:
        """Rank owning fp32 coordinate(s) x in [0, Lx): the same fp32 comparisons md_dd_select makes."""
        x = np.asarray(x, dtype=np.float32)
        r = np.searchsorted(self.bounds[1:], x, side="right")
        return np.minimum(r, self.nranks - 1).astype(np.int64)


def select_np(x, lo: float, hi: float) -> np.ndarray:
    """numpy twin of md_dd_select (fp32 comparisons, ascending index)."""
    x = np.asarray(x, dtype=np.float32)
    return np.nonzero((x >= np.float32(lo)) & (x < np.float32(hi)))[0]


def local_sets_np(pos, plan: SlabPlan, rank: int):
    """(owned, ghosts) index arrays of `rank` for wrapped positions pos[:, 0] -- the reference the tests hold the GPU path to."""
    x = np.asarray(pos, dtype=np.float32)[:, 0]
    own = plan.owner(x)
    owned = np.nonzero(own == rank)[0]
    if plan.nranks == 1:
        return owned, np.zeros(0, dtype=np.int64)
    L, R = plan.left(rank), plan.right(rank)
    zl = plan.zone_to_right(L)      # what the left neighbour sends to its right
    zr = plan.zone_to_left(R)
    from_left = np.nonzero((own == L) & (x >= np.float32(zl[0])) & (x < np.float32(zl[1])))[0]
    from_right = np.nonzero((own == R) & (x >= np.float32(zr[0])) & (x < np.float32(zr[1])))[0]
    return owned, np.concatenate([from_left, from_right])


# ------------------------------------------------------------------------------------------------
# transports: deliver every domain's (to_left, to_right) messages; a message is a list of 2-D tensors with equal rows
# ------------------------------------------------------------------------------------------------
class LocalTransport:
    """All domains live in this process (tests of the protocol on one GPU): deliveries are references."""

    def __init__(self, plan: SlabPlan):
        self.plan = plan

    def exchange(self, outgoing):
        """outgoing[rank] = (to_left, to_right)  ->  incoming[rank] = (from_left, from_right)."""
        P = self.plan.nranks
        return {r: (outgoing[self.plan.left(r)][1], outgoing[self.plan.right(r)][0]) for r in range(P)}

    def any_flag(self, flags) -> bool:
        return bool(max(flags.values()))


class DistTransport:
    """One domain per process, torch.distributed point-to-point: backend nccl moves device buffers GPU to GPU; with
    `stage_host` the messages go through host memory (backend gloo: CPU tests, or several processes sharing one GPU)."""

    def __init__(self, plan: SlabPlan, dist, device, stage_host: bool = False):
        self.plan, self.dist, self.device = plan, dist, device
        self.wire = "cpu" if stage_host else device        # where the buffers handed to torch.distributed live
        self.rank = dist.get_rank()

    def _sendrecv(self, send_to, send_msg, recv_from, like):
        import torch
        dist = self.dist
        n_out = torch.tensor([send_msg[0].shape[0] if send_msg else 0], dtype=torch.int64, device=self.wire)
        n_in = torch.zeros(1, dtype=torch.int64, device=self.wire)
        ops = [dist.P2POp(dist.isend, n_out, send_to), dist.P2POp(dist.irecv, n_in, recv_from)]
        for w in dist.batch_isend_irecv(ops):
            w.wait()
        n = int(n_in.item())
        recv = [torch.empty((n,) + tuple(t.shape[1:]), dtype=t.dtype, device=self.wire) for t in like]
        ops = []
        for t in send_msg:
            if t.shape[0] > 0:
                ops.append(dist.P2POp(dist.isend, t.contiguous().to(self.wire), send_to))
        for t in recv:
            if n > 0:
                ops.append(dist.P2POp(dist.irecv, t, recv_from))
        if ops:
            for w in dist.batch_isend_irecv(ops):
                w.wait()
        return [r.to(self.device) for r in recv]

    def exchange(self, outgoing):
        r = self.rank
        to_left, to_right = outgoing[r]
        L, R = self.plan.left(r), self.plan.right(r)
        # phase 1: everyone sends right and receives from the left; phase 2 the other way round (no deadlock for any P >= 2)
        from_left = self._sendrecv(R, to_right, L, to_right)
        from_right = self._sendrecv(L, to_left, R, to_left)
        return {r: (from_left, from_right)}

    def any_flag(self, flags) -> bool:
        import torch
        t = torch.tensor([int(max(flags.values()))], dtype=torch.int32, device=self.wire)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return bool(t.item())


# ------------------------------------------------------------------------------------------------
# one rank's domain on its GPU
# ------------------------------------------------------------------------------------------------
class Domain:
    """Owned particles (original ids 0 .. n_own-1) + ghosts (from the left neighbour, then from the right one).  The global
    id of a particle travels in pos.w as int32 bits (the library carries pos.w along untouched)."""

    def __init__(self, rank: int, plan: SlabPlan, n_global: int, rcut: float, skin: float, potential: dict, max_neigh: int,
                 device: str = "cuda:0", order: str = "hilbert", strategy: str = "vertex", variant: str = "smem"):
        import torch
        from .binding import dd_select
        self.torch, self.select = torch, dd_select
        self.rank, self.plan = rank, plan
        self.rigid = potential["kind"] in ("patchy", "patchy_pp")
        self.strategy, self.variant = strategy, variant
        # capacity = the global particle count: cell tables and candidate masks are sized by the global density
        self.sys = MDSystem(n_global, plan.box, rcut, skin, potential, max_neigh, device=device, order=order)
        self.device = self.sys.device
        self.arrays = ["pos", "vel"] + (["quat", "angmom"] if self.rigid else [])
        self.halo_arrays = ["pos"] + (["quat"] if self.rigid else [])
        self.n_own = 0
        self.n_from_left = self.n_from_right = 0
        self.idx_left = self.idx_right = None      # send lists (original ids of owned particles in the two halo zones)
        self.n_rebuilds = 0

    # ---- setup: the rank's share of the global initial state (host arrays in global id order; setup plumbing) ----
    def load_initial(self, pos, vel, quat=None, angmom=None):
        t = self.torch
        x = np.asarray(pos, dtype=np.float32)
        mine = np.nonzero(self.plan.owner(x[:, 0]) == self.rank)[0]
        p = x[mine].copy()
        p[:, 3] = mine.astype(np.int32).view(np.float32)            # global id in pos.w
        self.n_own = int(mine.shape[0])
        self.sys.resize(self.n_own)
        up = lambda a: t.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(self.device)
        self.sys.pos.copy_(up(p)); self.sys.vel.copy_(up(np.asarray(vel)[mine]))
        if self.rigid:
            self.sys.quat.copy_(up(np.asarray(quat)[mine])); self.sys.angmom.copy_(up(np.asarray(angmom)[mine]))

    # ---- rebuild, phase 1: wrap, then hand the particles that left the slab to the neighbours ----
    def migrate_out(self):
        s, plan, r = self.sys, self.plan, self.rank
        s.build_cells()                                             # wraps positions into the box (and reorders storage)
        own_pos = s.gather_ids("pos", first_id=0, n=self.n_own)     # owned particles in id order
        lo, hi = plan.slab(r)
        stay = self.select(own_pos, lo, hi)
        empty = own_pos[:0].to(self.torch.int32).reshape(0)
        if plan.nranks == 1:
            go_left = go_right = empty
        else:
            go_right = self.select(own_pos, *plan.slab(plan.right(r)))
            go_left = self.select(own_pos, *plan.slab(plan.left(r))) if plan.left(r) != plan.right(r) else empty
        if int(stay.shape[0] + go_left.shape[0] + go_right.shape[0]) != self.n_own:
            raise RuntimeError(f"rank {r}: a particle moved further than one slab between two rebuilds")
        pack = lambda idx: [s.gather_ids(a, ids=idx) for a in self.arrays]
        self._stay = pack(stay)
        return pack(go_left), pack(go_right)

    def migrate_in(self, from_left, from_right):
        t, s = self.torch, self.sys
        parts = [self._stay] + [m for m in (from_left, from_right) if m and m[0].shape[0] > 0]
        self.n_own = int(sum(p[0].shape[0] for p in parts))
        if self.n_own == 0:
            raise RuntimeError(f"rank {self.rank}: no particles left in the slab")
        s.resize(self.n_own)                                        # owned only, for the halo selection below
        for k, a in enumerate(self.arrays):
            getattr(s, a).copy_(t.cat([p[k] for p in parts], dim=0))
        s.vel[:, 3] = 0.0
        del self._stay

    # ---- rebuild, phase 2: the halo ----
    def halo_out(self):
        s, plan, r = self.sys, self.plan, self.rank
        if plan.nranks == 1:
            self.idx_left = self.idx_right = s.pos[:0, 0].to(self.torch.int32)
            return [], []
        self.idx_left = self.select(s.pos, *plan.zone_to_left(r))   # storage is in id order right after the bind
        self.idx_right = self.select(s.pos, *plan.zone_to_right(r))
        return ([s.gather_ids(a, ids=self.idx_left) for a in self.halo_arrays],
                [s.gather_ids(a, ids=self.idx_right) for a in self.halo_arrays])

    def halo_in(self, from_left, from_right):
        t, s = self.torch, self.sys
        nl = int(from_left[0].shape[0]) if from_left else 0
        nr = int(from_right[0].shape[0]) if from_right else 0
        self.n_from_left, self.n_from_right = nl, nr
        own = {a: getattr(s, a).clone() for a in self.arrays}       # md_resize keeps the rows, but be explicit
        s.resize(self.n_own + nl + nr)
        for a in self.arrays:
            getattr(s, a)[:self.n_own].copy_(own[a])
            getattr(s, a)[self.n_own:].zero_()
        for k, a in enumerate(self.halo_arrays):
            if nl:
                getattr(s, a)[self.n_own:self.n_own + nl].copy_(from_left[k])
            if nr:
                getattr(s, a)[self.n_own + nl:].copy_(from_right[k])
        s.set_active(self.n_own)
        s.build_cells(); s.build_verlet()
        s.forces(self.strategy, self.variant)
        self.n_rebuilds += 1

    # ---- one step ----
    def kick_drift(self, dt):
        self.sys.half_step(dt, "kick_drift")

    def refresh_out(self):
        s = self.sys
        if self.plan.nranks == 1:
            return [], []
        return ([s.gather_ids(a, ids=self.idx_left) for a in self.halo_arrays],
                [s.gather_ids(a, ids=self.idx_right) for a in self.halo_arrays])

    def refresh_in(self, from_left, from_right):
        s = self.sys
        for k, a in enumerate(self.halo_arrays):
            if self.n_from_left:
                s.scatter_ids(a, self.n_own, from_left[k])
            if self.n_from_right:
                s.scatter_ids(a, self.n_own + self.n_from_left, from_right[k])

    def flag(self) -> int:
        return self.sys.rebuild_flag()

    def forces(self):
        self.sys.forces(self.strategy, self.variant)

    def kick(self, dt):
        self.sys.half_step(dt, "kick")

    # ---- read-back (tests, output): owned rows in id order with their global ids ----
    def owned(self, array: str):
        a = self.sys.gather_ids(array, first_id=0, n=self.n_own).cpu().numpy()
        p = self.sys.gather_ids("pos", first_id=0, n=self.n_own).cpu().numpy()
        return p[:, 3].copy().view(np.int32), a

    def close(self):
        self.sys.close()


class DDSimulation:
    """The protocol over the domains of this process (one per process under torch.distributed; all of them with the
    in-process transport)."""

    def __init__(self, domains: List[Domain], transport):
        self.domains = {d.rank: d for d in domains}
        self.transport = transport
        self.steps = 0

    def rebuild(self):
        out = {r: d.migrate_out() for r, d in self.domains.items()}
        inc = self.transport.exchange(out)
        for r, d in self.domains.items():
            d.migrate_in(*inc[r])
        out = {r: d.halo_out() for r, d in self.domains.items()}
        inc = self.transport.exchange(out)
        for r, d in self.domains.items():
            d.halo_in(*inc[r])

    def step(self, dt):
        for d in self.domains.values():
            d.kick_drift(dt)
        inc = self.transport.exchange({r: d.refresh_out() for r, d in self.domains.items()})
        for r, d in self.domains.items():
            d.refresh_in(*inc[r])
        if self.transport.any_flag({r: d.flag() for r, d in self.domains.items()}):
            self.rebuild()                                   # ends with a force evaluation on the new lists
        else:
            for d in self.domains.values():
                d.forces()
        for d in self.domains.values():
            d.kick(dt)
        self.steps += 1

    def run(self, dt, nsteps):
        for _ in range(nsteps):
            self.step(dt)

    def energy(self):
        """(U, K_trans, K_rot) summed over the owned particles of the local domains (all-reduce it across processes)."""
        e = np.zeros(3)
        for d in self.domains.values():
            e += np.array(d.sys.energy())
        return tuple(e)

    def gather(self, array: str, n_global: int):
        """Rows of `array` of the local domains' owned particles placed at their global ids ([n_global, 4], NaN elsewhere)."""
        out = np.full((n_global, 4), np.nan, dtype=np.float32)
        for d in self.domains.values():
            gid, a = d.owned(array)
            out[gid] = a
        return out

    def close(self):
        for d in self.domains.values():
            d.close()
