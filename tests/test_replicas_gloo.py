"""world_size-2 CPU test (gloo) of the benchmark's multi-rank plumbing: replicas only, no data-path
collective; timing = max over ranks, work = sum over ranks."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1412_0659_b200.replicas import replica_seed, reduce_max_sum, whole_job_rate


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from nbody_inputs import plummer
        pos, _, _ = plummer(256, replica_seed(1002, rank))
        secs, units = (2.0, 100.0) if rank == 0 else (3.0, 50.0)
        mx, sm = reduce_max_sum([secs, units, float(pos.double().sum())])
        rate = whole_job_rate(secs, units)
        gathered = [None] * world
        dist.all_gather_object(gathered, float(pos.double().sum()))
        out.put((rank, mx, sm, rate, gathered))
    finally:
        dist.destroy_process_group()


def test_two_rank_replicas_reduce_max_time_sum_work():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, sm, rate, gathered in res:
        assert mx[0] == 3.0 and sm[1] == 150.0      # slowest rank's time, all ranks' work
        assert rate == 150.0 / 3.0
        assert gathered[0] != gathered[1]           # the two replicas are different particle sets
        assert abs(sm[2] - (gathered[0] + gathered[1])) < 1e-9


def test_single_process_is_identity():
    mx, sm = reduce_max_sum([1.5, 7.0])
    assert mx == [1.5, 7.0] and sm == [1.5, 7.0]
    assert whole_job_rate(2.0, 10.0) == 5.0
    assert replica_seed(1002, 0) == 1002 and replica_seed(1002, 3) != replica_seed(1002, 2)
