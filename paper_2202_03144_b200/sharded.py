"""One scan over several GPUs (reading R27 of DESIGN.md).

One process per GPU.  The frames are split into row bands (`shard_plan`); every rank holds the exit waves and
intensities of its own frames and drives the C ABI's `ptycho_shard_begin` / `ptycho_shard_end`; between the two this
module moves what has to cross GPUs with `torch.distributed` (NCCL on GPUs): the correction canvas on the object rows
two ranks both cover (neighbour send / receive of contiguous row blocks) and the probe sums (one all-reduce of 3 N^2
floats).  Nothing of the cycle's arithmetic is here except those additions of partial sums.

`LocalGroup` runs all shards of a plan in ONE process on one GPU, in lockstep and with the same exchange code, so that
the sharded path can be checked against the oracle on a single-GPU box (no rank ever waits for another rank's kernel).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


# ---------------------------------------------------------------------------------------------
# the plan: pure integer work on the positions (numpy only; checked bit-exactly in tests/)
# ---------------------------------------------------------------------------------------------
@dataclass
class ShardPlan:
    n: int                                  # frame size N
    H: int
    W: int
    world: int
    frames: list                            # per rank: indices (into the scan's position list) of its frames, ascending (y, x)
    rows: list                              # per rank: (row0, row1) = object rows its frames cover
    foreign: list                           # per rank: indices of the other ranks' frames that touch rows [row0, row1)
    exchange: list                          # per rank: [(peer, lo, hi)] = rows both cover, ascending peer
    owned: list                             # per rank: (lo, hi) rows it contributes to the stitched object (disjoint over ranks)
    total: int = 0
    meta: dict = field(default_factory=dict)


def shard_plan(pos, n: int, H: int, W: int, world: int) -> ShardPlan:
    """Row-band partition: frames sorted by (y, x), cut into `world` runs of (almost) equal length.  Bands keep the rows two
    ranks share few ("the overlapping size where the data is shared between multiple GPUs") and contiguous in
    memory, so that the exchange is a copy of whole row blocks."""
    pos = np.asarray(pos, np.int64).reshape(-1, 2)
    J = pos.shape[0]
    if world < 1 or J < world:
        raise ValueError("need at least one frame per rank")
    order = np.lexsort((pos[:, 1], pos[:, 0]))
    frames = [np.ascontiguousarray(a, np.int64) for a in np.array_split(order, world)]
    rows = [(int(pos[f, 0].min()), int(pos[f, 0].max()) + n) for f in frames]
    foreign, exchange, owned = [], [], []
    for r in range(world):
        lo, hi = rows[r]
        others = np.concatenate([frames[q] for q in range(world) if q != r]) if world > 1 else np.zeros(0, np.int64)
        touch = (pos[others, 0] < hi) & (pos[others, 0] + n > lo)
        foreign.append(np.sort(others[touch]))
        ex = []
        for q in range(world):
            if q == r:
                continue
            a, b = max(lo, rows[q][0]), min(hi, rows[q][1])
            if a < b:
                ex.append((q, a, b))
        exchange.append(ex)
        seen = max([rows[q][1] for q in range(r)], default=0)        # rows[.][0] ascends with the rank, so lower ranks cover [.., seen)
        owned.append((min(max(lo, seen), hi), hi))
    return ShardPlan(n, H, W, world, frames, rows, foreign, exchange, owned, J)


# ---------------------------------------------------------------------------------------------
# communication: torch.distributed (NCCL / gloo), or the in-process mailbox of LocalGroup
# ---------------------------------------------------------------------------------------------
class DistComm:
    """torch.distributed plumbing: batched neighbour send/receive and all-reduce on the default (or a given) group."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def sendrecv(self, sends, recvs):
        """sends / recvs: [(peer, contiguous tensor)].  Returns when the receives have landed."""
        d = self.dist
        ops = [d.P2POp(d.isend, t, p, self.group) for p, t in sends] + [d.P2POp(d.irecv, t, p, self.group) for p, t in recvs]
        if ops:
            for req in d.batch_isend_irecv(ops):
                req.wait()

    def all_reduce(self, t):
        self.dist.all_reduce(t, group=self.group)
        return t


class HaloExchange:
    """Adds, on the rows two ranks both cover, every other rank's part of a row-major canvas into this rank's (a1-a9 leave
    partial overlap sums; a10 needs the totals).  Works on any torch tensor whose first axis is the object row (CUDA views of
    the library's workspace, or CPU tensors in the gloo test)."""

    def __init__(self, plan: ShardPlan, rank: int):
        self.plan, self.rank = plan, rank
        self.peers = plan.exchange[rank]
        self._stage = None

    def outgoing(self, canvas):
        return [(p, canvas[lo:hi]) for p, lo, hi in self.peers]                 # contiguous row blocks: sent in place

    def staging(self, canvas):
        if not self.peers:
            return []
        if self._stage is None or self._stage[0].dtype != canvas.dtype or self._stage[0].device != canvas.device:
            self._stage = [canvas.new_empty((hi - lo,) + tuple(canvas.shape[1:])) for _, lo, hi in self.peers]
        return [(p, buf) for (p, _, _), buf in zip(self.peers, self._stage)]

    def accumulate(self, canvas, received):
        """received: [(peer, tensor)] in the order of self.peers (ascending peer): one fixed order of additions."""
        for (p, lo, hi), (q, buf) in zip(self.peers, received):
            assert p == q
            canvas[lo:hi] += buf

    def run(self, canvas, comm: DistComm):
        recvs = self.staging(canvas)
        if not recvs:
            return
        comm.sendrecv(self.outgoing(canvas), recvs)                             # the sends read the canvas before anything is added
        self.accumulate(canvas, recvs)


def stitch_rows(plan: ShardPlan, rank: int, obj_local, fill):
    """This rank's term of the stitched object: its owned rows of obj_local, zero elsewhere; rank 0 also brings the rows no
    frame covers (from `fill`, the initial object).  The sum of the terms over ranks is the object (disjoint supports)."""
    out = obj_local.new_zeros(obj_local.shape) if hasattr(obj_local, "new_zeros") else np.zeros_like(obj_local)
    lo, hi = plan.owned[rank]
    out[lo:hi] = obj_local[lo:hi]
    if rank == 0:
        covered = np.zeros(plan.H, bool)
        for a, b in plan.owned:
            covered[a:b] = True
        idx = np.nonzero(~covered)[0]
        if len(idx):
            if not isinstance(out, np.ndarray):
                import torch
                idx = torch.as_tensor(idx, device=out.device)
            out[idx] = fill[idx]
    return out


# ---------------------------------------------------------------------------------------------
# one shard = one C-ABI context
# ---------------------------------------------------------------------------------------------
class ShardedPtycho:
    """Rank `rank` of a scan split by `plan`.  intensities_local: the frames plan.frames[rank], in that order."""

    def __init__(self, plan: ShardPlan, rank: int, obj, probe, pos, intensities_local, comm=None, device="cuda:0", **params):
        import torch
        from . import binding
        self.plan, self.rank, self.comm = plan, rank, comm
        self._torch = torch
        pos = np.ascontiguousarray(np.asarray(pos).reshape(-1, 2), np.int32)
        mine = plan.frames[rank]
        assert intensities_local.shape[0] == len(mine)
        par = binding.default_params(shard_total_pos=plan.total, foreign_pos=pos[plan.foreign[rank]], **params)
        self.core = binding.Ptycho(obj, probe, pos[mine], intensities_local, par, device=device)
        self.buf = self.core.shard_buffers()
        assert (self.buf["row0"], self.buf["row1"]) == plan.rows[rank]
        self.halo = HaloExchange(plan, rank)
        self._obj0 = obj
        self._sum_I_shared = False
        if comm is not None:
            comm.all_reduce(self.buf["sum_I"])                              # the error's denominator is the scan's (C3)
            self._sum_I_shared = True

    # the three steps of an iteration; LocalGroup calls them in lockstep, iterate() in sequence
    def begin(self):
        assert self._sum_I_shared, "sum_I has not been summed over the shards"
        self.core.shard_begin()

    def exchange(self):
        self.halo.run(self.buf["c_canvas"], self.comm)
        self.comm.all_reduce(self.buf["probe_sums"])

    def end(self):
        self.core.shard_end()

    def iterate(self, n_iters: int = 1):
        for _ in range(n_iters):
            self.begin()
            self.exchange()
            self.end()
        return self

    # results (collective calls: every rank must make them)
    def fetch_object(self):
        """The stitched object, on every rank."""
        torch = self._torch
        O = torch.from_numpy(self.core.fetch_object()).to(self.core.device)
        fill = torch.as_tensor(np.asarray(self._obj0, np.complex64) if isinstance(self._obj0, np.ndarray) else self._obj0).to(self.core.device)
        term = torch.view_as_real(stitch_rows(self.plan, self.rank, O, fill)).contiguous()
        self.comm.all_reduce(term)
        return torch.view_as_complex(term).cpu().numpy()

    def fetch_probe(self):
        return self.core.fetch_probe()                                      # identical on every rank (the sums were all-reduced)

    def fetch_error(self):
        torch = self._torch
        e = torch.from_numpy(self.core.fetch_error()).to(self.core.device)
        self.comm.all_reduce(e)
        return e.cpu().numpy()

    def fetch_exit_waves(self, idx=None):
        """Exit waves of this rank's frames (local indices into plan.frames[rank])."""
        return self.core.fetch_exit_waves(idx)

    def destroy(self):
        self.core.destroy()


class LocalGroup:
    """All shards of a plan in one process on one GPU, stepped in lockstep with the exchange done through a mailbox: the
    single-GPU stand-in for N ranks (tests, smoke).  The data path is the one of the distributed run -- the same
    ptycho_shard_begin / _end calls, the same HaloExchange code, the same order of additions."""

    def __init__(self, plan: ShardPlan, obj, probe, pos, intensities, device="cuda:0", **params):
        import torch
        self._torch, self.plan = torch, plan
        self.shards = [ShardedPtycho(plan, r, obj, probe, pos, intensities[plan.frames[r]], comm=None, device=device, **params)
                       for r in range(plan.world)]
        total = sum(s.buf["sum_I"].clone() for s in self.shards)
        for s in self.shards:
            s.buf["sum_I"].copy_(total)
            s._sum_I_shared = True
        self._obj0 = obj

    def iterate(self, n_iters: int = 1):
        torch = self._torch
        for _ in range(n_iters):
            for s in self.shards:
                s.begin()
            # mailbox: every rank's outgoing blocks are copied out before any rank adds (what send / receive guarantees)
            box = {}
            for s in self.shards:
                for p, t in s.halo.outgoing(s.buf["c_canvas"]):
                    box[(s.rank, p)] = t.clone()
            for s in self.shards:
                s.halo.accumulate(s.buf["c_canvas"], [(p, box[(p, s.rank)]) for p, _, _ in s.halo.peers])
            tot = torch.stack([s.buf["probe_sums"] for s in self.shards]).sum(0)
            for s in self.shards:
                s.buf["probe_sums"].copy_(tot)
                s.end()
        return self

    def fetch_object(self):
        O = None
        fill = np.asarray(self._obj0, np.complex64)
        for s in self.shards:
            term = stitch_rows(self.plan, s.rank, s.core.fetch_object(), fill)
            O = term if O is None else O + term
        return O

    def fetch_probe(self):
        return self.shards[0].core.fetch_probe()

    def fetch_error(self):
        return sum(s.core.fetch_error() for s in self.shards)

    def fetch_exit_waves(self):
        """All exit waves in the scan's frame order."""
        s0 = self.shards[0].core
        out = np.empty((self.plan.total, s0.K, s0.n, s0.n), np.complex64)
        for s in self.shards:
            out[self.plan.frames[s.rank]] = s.core.fetch_exit_waves()
        return out

    def destroy(self):
        for s in self.shards:
            s.destroy()
