"""world_size-2 CPU test (gloo) of the host side of the sharded force pass (paper_1412_0659_b200/sharded.py,
DESIGN.md §7): set-up order, exchange of the result-buffer handles, the begin -> barrier -> end sequence and
the reduced interaction totals.  The CUDA context is replaced by a stand-in that records the calls and
emulates the peer stores through files, so the test also shows that no rank runs its second half before
every rank has finished its first half."""
import os
import socket
import time

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1412_0659_b200.sharded import ShardedTree


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


class StandInTree:
    """Records the call sequence; 'peer stores' are files in a directory every rank can see."""

    def __init__(self, rank, tmp):
        self.rank, self.tmp, self.calls, self.peers, self.passes = rank, tmp, [], {}, 0
        self.device = "cpu"

    def reserve(self, n): self.calls.append(("reserve", n))
    def shard_config(self, rank, world): self.calls.append(("config", rank, world)); self.world = world
    def shard_export(self): self.calls.append(("export",)); return bytes([self.rank + 1]) * 128
    def shard_attach(self, r, h): self.calls.append(("attach", r)); self.peers[r] = h
    def build(self, pos, mass): self.calls.append(("build",))
    def set_velocity(self, v): self.calls.append(("vel",))

    def _begin(self, what="pass"):
        self.passes += 1
        if self.rank == 1:
            time.sleep(0.5)  # a slow rank: the others must wait for it at the barrier
        with open(os.path.join(self.tmp, f"{what}{self.passes}_from{self.rank}"), "w") as f:
            f.write("stored")

    def _end(self, what="pass", tag="end_saw_all"):
        # every rank's preceding part must be complete: its "store" is visible
        seen = [os.path.exists(os.path.join(self.tmp, f"{what}{self.passes}_from{r}")) for r in range(self.world)]
        self.calls.append((tag, all(seen)))

    def force_begin(self, theta, eps): self.calls.append(("force_begin",)); self._begin()
    def force_end(self, acc=None, pot=None): self._end()
    def leapfrog_begin(self, dt): self.calls.append(("leapfrog_begin",)); self._begin("sorted")   # sorted run "stored"

    def leapfrog_mid(self):
        self._end("sorted", "mid_saw_all")      # reads every rank's sorted run: needs the first barrier
        self.passes -= 1
        self._begin("pass")                     # the walk "stores" its results

    def leapfrog_end(self): self._end()
    def stats(self): return {"walk": 1.0 + self.rank}, 100 * (self.rank + 1), 7 * (self.rank + 1)
    def shard_range(self): return (self.rank, self.rank + 1, 64 * self.rank, 64 * (self.rank + 1))
    def close(self): self.calls.append(("close",))


def _worker(rank, world, port, tmp, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        st = ShardedTree(StandInTree(rank, tmp))
        st.connect(1000)
        st.build(None, None)
        st.set_velocity(None)
        st.force(0.4, 0.01)
        st.leapfrog(1e-3)
        ms, pp, pc = st.stats()
        st.close()
        out.put((rank, st.tree.calls, sorted(st.tree.peers.items()), ms, pp, pc))
    finally:
        dist.destroy_process_group()


def test_two_rank_sharded_sequence(tmp_path):
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, str(tmp_path), q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, calls, peers, ms, pp, pc in res:
        names = [c[0] for c in calls]
        assert names[:4] == ["reserve", "config", "export", "attach"]           # set-up order of include/tree.h
        assert calls[1] == ("config", rank, world)
        assert peers == [(1 - rank, bytes([2 - rank]) * 128)]                     # the OTHER rank's handle, under its rank
        assert names[4:] == ["build", "vel", "force_begin", "end_saw_all", "leapfrog_begin", "mid_saw_all", "end_saw_all",
                             "close"]
        assert all(c[1] for c in calls if c[0] in ("end_saw_all", "mid_saw_all"))  # a barrier sits between the parts
        assert (pp, pc) == (300, 21)                                             # totals are summed over the ranks
        assert ms["walk"] == 1.0 + rank                                          # times stay per rank


def test_single_process_needs_no_group():
    st = ShardedTree(StandInTree(0, "/nonexistent"))
    assert (st.rank, st.world) == (0, 1)
    st.connect(10)
    assert [c[0] for c in st.tree.calls] == ["reserve", "config"]  # nothing to exchange
    _, pp, pc = st.stats()
    assert (pp, pc) == (100, 7)
