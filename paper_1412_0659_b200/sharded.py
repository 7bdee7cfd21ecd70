"""Sharded force pass over the GPUs of one NVLink / NVSwitch node (include/tree.h "sharded force pass",
DESIGN.md §7; PAPER.md L81-125 is the paper's multi-GPU scheme this replaces on such a node).

Every rank (one process per GPU, ``torch.distributed``) holds all N particles and builds the same
tree; rank r walks one contiguous, cost-balanced range of the Peano-Hilbert-sorted groups
 and its walk kernel stores the results straight into every rank's result
buffers (peer stores over NVLink).  In a leapfrog step the sort is cut as well, by key range: every rank sorts its
own range and stores the sorted run into every rank.  The only collectives are the barriers between the parts of a
pass / step: one 8-byte all-reduce each on the stream the context works on.

This module is host logic only: set-up (exchange of the IPC handles), the begin / barrier / end
sequence, the reduced totals.  It drives any object with the ``Tree`` methods it names, so the
sequence is covered on CPU with the gloo backend and a stand-in tree (tests/test_sharded_gloo.py).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def _world(group=None):
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(group), dist.get_world_size(group)
    return 0, 1


class ShardedTree:
    """``tree`` is this rank's ``Tree`` (or a stand-in with the same methods)."""

    def __init__(self, tree, group=None, device=None):
        self.tree = tree
        self.group = group
        self.rank, self.world = _world(group)
        self.device = device if device is not None else getattr(tree, "device", "cpu")
        self.connected = False
        self.totals = None  # (n_pp, n_pc) of the last pass, summed over ranks

    # -- set-up: reserve, tell the context its rank, exchange and attach the result-buffer handles
    def connect(self, n_max: int):
        t = self.tree
        t.reserve(int(n_max))
        t.shard_config(self.rank, self.world)
        if self.world > 1:
            mine = t.shard_export()
            handles = [None] * self.world
            dist.all_gather_object(handles, mine, group=self.group)
            err = None
            try:
                for r, h in enumerate(handles):
                    if r != self.rank:
                        t.shard_attach(r, h)
            except Exception as e:  # e.g. GPUs that are not peer-capable
                err = e
            # every rank learns whether all attached (also: nobody starts a pass before everybody has attached)
            if self._sum([0 if err else 1])[0] != self.world:
                t.shard_config(0, 1)
                raise RuntimeError(f"sharded set-up failed on at least one rank (this rank: {err})")
        self.connected = True

    # -- the exchange step: one all-reduce, enqueued on the stream the context works on.  It carries no
    #    payload the pass needs: it orders every rank's peer stores before anybody's second half.
    def _barrier(self):
        if self.world > 1:
            if getattr(self, "_flag", None) is None:
                self._flag = torch.zeros(1, dtype=torch.int64, device=self.device)
            raw = getattr(self.tree, "stream", None)
            if raw is None:  # a stand-in tree (CPU tests of the host sequence): nothing to order on a device
                dist.all_reduce(self._flag, op=dist.ReduceOp.SUM, group=self.group)
                return
            # A real context: the all-reduce must be ordered on the stream the context's kernels run on, whatever
            # torch's current stream is, and only a device-side (NCCL) collective orders anything there.
            if dist.get_backend(self.group) != "nccl":
                raise RuntimeError("ShardedTree needs the nccl backend: its barrier must be a collective on the GPU stream")
            s = torch.cuda.ExternalStream(raw, device=self.device) if raw else torch.cuda.default_stream(self.device)
            with torch.cuda.stream(s):
                dist.all_reduce(self._flag, op=dist.ReduceOp.SUM, group=self.group)

    def _sum(self, values):
        v = torch.tensor([int(x) for x in values], dtype=torch.int64, device=self.device)
        if self.world > 1:
            dist.all_reduce(v, op=dist.ReduceOp.SUM, group=self.group)
        return [int(x) for x in v.tolist()]

    # -- the path
    def build(self, pos, mass):
        assert self.connected, "call connect(n_max) first"
        self.tree.build(pos, mass)

    def set_velocity(self, vel):
        self.tree.set_velocity(vel)

    def force(self, theta: float, eps: float, acc=None, pot=None):
        self.tree.force_begin(theta, eps)
        self._barrier()
        self.tree.force_end(acc, pot)

    def leapfrog(self, dt: float):
        self.tree.leapfrog_begin(dt)   # kick, drift, keys; this rank's key range sorted and stored into every rank
        self._barrier()
        self.tree.leapfrog_mid()       # gather, octree, moments, walk of this rank's groups (results into every rank)
        self._barrier()
        self.tree.leapfrog_end()       # kick

    def stats(self):
        """Per-phase times of this rank; interaction totals summed over ranks (each rank counts its range)."""
        ms, pp, pc = self.tree.stats()
        self.totals = tuple(self._sum([pp, pc]))
        return ms, self.totals[0], self.totals[1]

    def shard_range(self):
        return self.tree.shard_range()

    def close(self):
        if self.world > 1:
            self._barrier()  # no peer may still be storing into buffers that are about to be freed
        self.tree.close()


def connect_local(trees):
    """Several contexts of ONE process (one per GPU, or several on one GPU for the parity tests):
    context r becomes rank r of len(trees); all must have reserved the same N."""
    world = len(trees)
    for r, t in enumerate(trees):
        t.shard_config(r, world)
    for r, t in enumerate(trees):
        for q, p in enumerate(trees):
            if q != r:
                t.shard_attach_local(q, p)


def force_local(trees, theta, eps, outs=None):
    """One sharded pass over contexts of one process; the barrier is the stream order / a device sync."""
    for t in trees:
        t.force_begin(theta, eps)
    torch.cuda.synchronize()
    for i, t in enumerate(trees):
        acc, pot = outs[i] if outs else (None, None)
        t.force_end(acc, pot)


def leapfrog_local(trees, dt):
    for t in trees:
        t.leapfrog_begin(dt)
    torch.cuda.synchronize()
    for t in trees:
        t.leapfrog_mid()
    torch.cuda.synchronize()
    for t in trees:
        t.leapfrog_end()
