"""GPU parity of the sharded force pass (include/tree.h "sharded force pass"): `world`
contexts share one pass, each walking one contiguous cost-balanced range of the PH-sorted groups
 and storing its results into every context's buffers.  One GPU is enough to
check the path: the contexts live in one process on cuda:0 and their kernels run one after the other
(none waits for another); across GPUs the same stores go over NVLink.  Every context must end up with
the complete result, equal to the oracle's within 1e-5 and with bit-exact interaction counts."""
import numpy as np
import pytest
import torch

import oracle
from nbody_inputs import plummer, milky_way
from paper_1412_0659_b200 import Tree, TreeError
from paper_1412_0659_b200.sharded import connect_local, force_local, leapfrog_local

pytestmark = pytest.mark.gpu
TOL = 1e-5


def _make(world, n, leaf=16, group=64):
    trees = [Tree(device=0, leaf_size=leaf, group_size=group) for _ in range(world)]
    for t in trees:
        t.reserve(n)
    connect_local(trees)
    return trees


def _close(trees):
    torch.cuda.synchronize()
    for t in trees:
        t.close()


@pytest.mark.parametrize("model,n,seed,world", [
    ("plummer", 20011, 11, 2),   # ragged last group
    ("plummer", 16384, 1001, 3), # BASELINE config 1, three ranks
    ("mw", 100000, 3, 4),        # deep, uneven tree: cost balance differs strongly from count balance
    ("plummer", 300, 4, 8),      # fewer groups than ranks x 4: some ranks own no or one group
])
def test_sharded_pass_equals_oracle_on_every_rank(model, n, seed, world):
    theta, eps = 0.4, 0.01
    pos, _, mass = (plummer if model == "plummer" else milky_way)(n, seed, with_vel=False)
    dpos, dmass = pos.cuda(), mass.cuda()
    trees = _make(world, n)
    outs = [(torch.zeros((n, 3), device="cuda"), torch.zeros(n, device="cuda")) for _ in range(world)]
    for t in trees:
        t.build(dpos, dmass)
    force_local(trees, theta, eps, outs)
    torch.cuda.synchronize()
    ot = oracle.Tree(pos.numpy(), mass.numpy())
    oacc, opot, onpp, onpc = ot.force(theta, eps)
    # the ranges tile the groups in rank order
    ranges = [t.shard_range() for t in trees]
    assert ranges[0][0] == 0 and ranges[-1][1] == ot.n_groups
    for a, b in zip(ranges[:-1], ranges[1:]):
        assert a[1] == b[0] and a[3] == b[2]
    assert all(r[0] <= r[1] for r in ranges)
    # cost balance: no rank above twice its fair share when it owns more than a few groups
    cost = 13.0 * onpp + 37.0 * onpc
    if ot.n_groups >= 32 * world:
        shares = [cost[r[0]:r[1]].sum() / cost.sum() for r in ranges]
        assert max(shares) < 2.0 / world, shares
    tot_pp = tot_pc = 0
    for t, (acc, pot) in zip(trees, outs):
        cnt = t.debug("counts")  # peers stored their groups' counts here
        assert np.array_equal(cnt[:, 0], onpp) and np.array_equal(cnt[:, 1], onpc)
        a = acc.cpu().numpy().astype(np.float64); p = pot.cpu().numpy().astype(np.float64)
        rel = np.linalg.norm(a - oacc, axis=1) / np.linalg.norm(oacc, axis=1)
        prel = np.abs(p - opot) / np.abs(opot)
        assert rel.max() <= TOL and prel.max() <= TOL, (rel.max(), prel.max())
        _, pp, pc = t.stats()
        tot_pp += pp; tot_pc += pc
    gs = np.minimum(ot.group_size, ot.n - ot.group_size * np.arange(ot.n_groups))
    assert tot_pp == int((onpp.astype(np.int64) * gs).sum()) and tot_pc == int((onpc.astype(np.int64) * gs).sum())
    # every rank holds the same bits
    for acc, pot in outs[1:]:
        assert torch.equal(acc, outs[0][0]) and torch.equal(pot, outs[0][1])
    _close(trees)


@pytest.mark.parametrize("leaf,group", [(16, 32), (8, 128)])
def test_sharded_pass_other_group_and_leaf_sizes(leaf, group):
    n, theta, eps, world = 25013, 0.5, 0.02, 3
    pos, _, mass = plummer(n, 17, with_vel=False)
    trees = _make(world, n, leaf=leaf, group=group)
    acc = torch.zeros((n, 3), device="cuda"); pot = torch.zeros(n, device="cuda")
    for t in trees:
        t.build(pos.cuda(), mass.cuda())
    force_local(trees, theta, eps, [(acc, pot)] + [(None, None)] * (world - 1))
    torch.cuda.synchronize()
    ot = oracle.Tree(pos.numpy(), mass.numpy(), leaf_size=leaf, group_size=group)
    oacc, opot, onpp, onpc = ot.force(theta, eps)
    for t in trees:
        cnt = t.debug("counts")
        assert np.array_equal(cnt[:, 0], onpp) and np.array_equal(cnt[:, 1], onpc)
    a = acc.cpu().numpy().astype(np.float64); p = pot.cpu().numpy().astype(np.float64)
    assert (np.linalg.norm(a - oacc, axis=1) / np.linalg.norm(oacc, axis=1)).max() <= TOL
    assert (np.abs(p - opot) / np.abs(opot)).max() <= TOL
    _close(trees)


def test_sharded_leapfrog_matches_single_context_and_ranks_agree_bitwise():
    n, theta, eps, dt, steps, world = 30011, 0.4, 0.01, 1e-3, 4, 3
    pos, vel, mass = plummer(n, 21)
    dpos, dvel, dmass = pos.cuda(), vel.cuda(), mass.cuda()
    single = Tree(device=0)
    single.build(dpos, dmass); single.set_velocity(dvel); single.force(theta, eps)
    trees = _make(world, n)
    for t in trees:
        t.build(dpos, dmass); t.set_velocity(dvel)
    force_local(trees, theta, eps)
    for _ in range(steps):
        single.leapfrog(dt)
        leapfrog_local(trees, dt)  # steps after the first schedule and partition by the previous pass's counts
    torch.cuda.synchronize()

    def state(t):
        p = torch.empty((n, 3), device="cuda"); v = torch.empty((n, 3), device="cuda")
        a = torch.empty((n, 3), device="cuda"); ph = torch.empty(n, device="cuda")
        t.get_state(p, v, a, ph)
        return p, v, a, ph

    ref = state(single)
    sts = [state(t) for t in trees]
    for st in sts[1:]:
        for x, y in zip(st, sts[0]):
            assert torch.equal(x, y)  # identical inputs, identical tree, the same stored results
    for x, y in zip(sts[0], ref):
        d = (x.double() - y.double()).abs().max().item()
        assert d <= 2e-6 * y.double().abs().max().item(), d  # a few partial sums are ordered differently
    # the partition follows the previous pass's costs: ranges still tile the groups
    ranges = [t.shard_range() for t in trees]
    assert ranges[0][0] == 0 and ranges[-1][1] == (n + 63) // 64
    assert all(a[1] == b[0] for a, b in zip(ranges[:-1], ranges[1:]))
    single.close(); _close(trees)


def test_sharded_call_order_errors():
    n = 4096
    pos, _, mass = plummer(n, 5, with_vel=False)
    t = Tree(device=0)
    with pytest.raises(TreeError) as e:
        t.shard_config(0, 2)          # needs tree_reserve first
    assert e.value.code == -4
    t.reserve(n)
    with pytest.raises(TreeError):
        t.shard_config(2, 2)          # rank out of range
    t.shard_config(0, 2)
    t.build(pos.cuda(), mass.cuda())
    with pytest.raises(TreeError) as e:
        t.force(0.4, 0.01)            # cannot contain the barrier
    assert e.value.code == -4
    with pytest.raises(TreeError) as e:
        t.force_begin(0.4, 0.01)      # peer 1 not attached
    assert e.value.code == -4
    big = plummer(2 * n, 5, with_vel=False)
    with pytest.raises(TreeError) as e:
        t.build(big[0].cuda(), big[2].cuda())  # beyond the reserved capacity: would invalidate exported buffers
    assert e.value.code == -4
    h = t.shard_export()
    assert len(h) == 128 and any(h)
    with pytest.raises(TreeError):
        t.force_end()                 # no pass open
    t.shard_config(0, 1)              # back to one context
    t.build(pos.cuda(), mass.cuda())
    t.force(0.4, 0.01)
    # begin / end on one context is tree_force in two halves
    acc = torch.empty((n, 3), device="cuda"); acc2 = torch.empty((n, 3), device="cuda")
    t.force(0.4, 0.01, acc)
    t.force_begin(0.4, 0.01)
    with pytest.raises(TreeError):
        t.force_begin(0.4, 0.01)      # already open
    t.force_end(acc2)
    assert torch.equal(acc, acc2)
    t.close()


def test_sharded_bench_size_config2_sampled_against_oracle():
    """BASELINE config 2 (Plummer N = 1,048,576), the size `bench.py --sharded` runs, on 4 contexts: interaction counts of
    every group equal the single-context pass (itself compared with the oracle at this size in
    test_bench_size_sampled_parity_config2); forces against the oracle on every 64th group within 1e-5."""
    from nbody_inputs import config
    cfg, pos, vel, mass = config(1, with_vel=False)
    n, world = cfg["n"], 4
    dpos, dmass = pos.cuda(), mass.cuda()
    single = Tree(device=0)
    single.build(dpos, dmass); single.force(cfg["theta"], cfg["eps"])
    ref_cnt = single.debug("counts")
    single.close()
    trees = _make(world, n)
    acc = torch.zeros((n, 3), device="cuda"); pot = torch.zeros(n, device="cuda")
    for t in trees:
        t.build(dpos, dmass)
    force_local(trees, cfg["theta"], cfg["eps"], [(acc, pot)] + [(None, None)] * (world - 1))
    torch.cuda.synchronize()
    ranges = [t.shard_range() for t in trees]
    assert ranges[0][0] == 0 and ranges[-1][1] == (n + 63) // 64
    assert all(a[1] == b[0] for a, b in zip(ranges[:-1], ranges[1:]))
    assert min(r[1] - r[0] for r in ranges) > 0
    for t in trees:
        assert np.array_equal(t.debug("counts"), ref_cnt)
    ot = oracle.Tree(pos.numpy(), mass.numpy())
    _, order, _ = ot.keys()
    stride = 64
    oacc, opot, onpp, onpc = ot.force(cfg["theta"], cfg["eps"], g0=7, stride=stride)
    gsel = np.arange(7, ot.n_groups, stride)
    assert np.array_equal(ref_cnt[gsel, 0], onpp[gsel]) and np.array_equal(ref_cnt[gsel, 1], onpc[gsel])
    sel = np.concatenate([order[64 * g: 64 * g + 64] for g in gsel])
    a = acc.cpu().numpy().astype(np.float64)[sel]; p = pot.cpu().numpy().astype(np.float64)[sel]
    rel = np.linalg.norm(a - oacc[sel], axis=1) / np.linalg.norm(oacc[sel], axis=1)
    assert rel.max() <= TOL, rel.max()
    assert (np.abs(p - opot[sel]) / np.abs(opot[sel])).max() <= TOL
    _close(trees)


def test_contexts_with_different_pass_histories_share_a_pass():
    # The result buffers are double-buffered by pass parity and peers store into the same parity: a context that has
    # already run unsharded passes (odd pass count) must still pair with a fresh one (tree_shard_config restarts the count).
    n, theta, eps = 12000, 0.4, 0.01
    pos, _, mass = plummer(n, 5, with_vel=False)
    dpos, dmass = pos.cuda(), mass.cuda()
    a, b = Tree(device=0), Tree(device=0)
    a.build(dpos, dmass); a.force(theta, eps)          # one unsharded pass on a only: a.pass = 1, b.pass = 0
    for t in (a, b):
        t.reserve(n)
    connect_local([a, b])
    outs = [(torch.zeros((n, 3), device="cuda"), torch.zeros(n, device="cuda")) for _ in range(2)]
    for t in (a, b):
        t.build(dpos, dmass)
    for _ in range(3):                                  # odd and even parities
        force_local([a, b], theta, eps, outs)
        torch.cuda.synchronize()
        assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])
    ot = oracle.Tree(pos.numpy(), mass.numpy())
    oacc, opot, onpp, onpc = ot.force(theta, eps)
    for t, (acc, pot) in zip((a, b), outs):
        cnt = t.debug("counts")
        assert np.array_equal(cnt[:, 0], onpp) and np.array_equal(cnt[:, 1], onpc)
        rel = np.linalg.norm(acc.cpu().numpy().astype(np.float64) - oacc, axis=1) / np.linalg.norm(oacc, axis=1)
        assert rel.max() <= TOL
    # back to one context each: the unsharded call works again and gives the same forces
    a.shard_config(0, 1)
    acc1 = torch.zeros((n, 3), device="cuda"); pot1 = torch.zeros(n, device="cuda")
    a.force(theta, eps, acc1, pot1)
    torch.cuda.synchronize()
    rel = np.linalg.norm(acc1.cpu().numpy().astype(np.float64) - oacc, axis=1) / np.linalg.norm(oacc, axis=1)
    assert rel.max() <= TOL
    _close([a, b])


_IPC_WORKER = r"""
import os, sys
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, os.environ["BH_ROOT"])
from nbody_inputs import plummer
from paper_1412_0659_b200 import Tree
from paper_1412_0659_b200.sharded import ShardedTree
torch.cuda.set_device(0)
dist.init_process_group("gloo")   # handle exchange only; the barrier between the two halves is explicit below
rank, world = dist.get_rank(), dist.get_world_size()
n, theta, eps, dt = 30011, 0.4, 0.01, 0.002
pos, vel, mass = plummer(n, 13)
t = Tree(device=0)
t.reserve(n); t.shard_config(rank, world)
handles = [None] * world
dist.all_gather_object(handles, t.shard_export())
for r, h in enumerate(handles):
    if r != rank:
        t.shard_attach(r, h)            # cudaIpcOpenMemHandle on the other PROCESS's result slab
dist.barrier()
def host_barrier():
    torch.cuda.synchronize(); dist.barrier()   # both ranks share one GPU: a device collective could deadlock them
acc = torch.zeros((n, 3), device="cuda"); pot = torch.zeros(n, device="cuda")
t.build(pos.cuda(), mass.cuda()); t.set_velocity(vel.cuda())
t.force_begin(theta, eps); host_barrier(); t.force_end(acc, pot)
for _ in range(2):
    t.leapfrog_begin(dt); host_barrier(); t.leapfrog_mid(); host_barrier(); t.leapfrog_end()
p = torch.empty((n, 3), device="cuda"); a = torch.empty((n, 3), device="cuda"); ph = torch.empty(n, device="cuda")
t.get_state(p, None, a, ph); torch.cuda.synchronize()
lo, hi, _, _ = t.shard_range()
np.savez(os.environ["BH_OUT"] + f".{rank}.npz", acc0=acc.cpu().numpy(), pot0=pot.cpu().numpy(), p=p.cpu().numpy(),
         a=a.cpu().numpy(), ph=ph.cpu().numpy(), counts=t.debug("counts"), rng=np.array([lo, hi]))
host_barrier()                          # nobody unmaps while the peer may still store
t.close()
dist.destroy_process_group()
"""


def test_cross_process_ipc_sharded_pass_two_processes_one_gpu(tmp_path):
    # tree_shard_export / tree_shard_attach across PROCESSES (cudaIpcGetMemHandle / cudaIpcOpenMemHandle): two
    # processes on cuda:0 share a force pass and two leapfrog steps; each process's kernel stores its groups into the
    # other process's buffers.  Both must end with the complete result, bit-identical to each other and to
    # connect_local contexts in one process, counts bit-exact against the oracle.
    import os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "ipc_worker.py"; script.write_text(_IPC_WORKER)
    env = dict(os.environ, BH_ROOT=root, BH_OUT=str(tmp_path / "out"), MASTER_ADDR="127.0.0.1", MASTER_PORT="29533",
               WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r)), stdout=subprocess.PIPE,
                              stderr=subprocess.STDOUT, text=True) for r in range(2)]
    outs = [p.communicate(timeout=600)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs), "\n".join(outs)
    r0, r1 = (np.load(str(tmp_path / f"out.{r}.npz")) for r in range(2))
    for k in ("acc0", "pot0", "p", "a", "ph", "counts"):
        assert np.array_equal(r0[k], r1[k]), k
    assert r0["rng"][0] == 0 and r0["rng"][1] == r1["rng"][0] and r1["rng"][1] == len(r0["counts"])
    # the same run with two contexts of ONE process
    n, theta, eps, dt = 30011, 0.4, 0.01, 0.002
    pos, vel, mass = plummer(n, 13)
    trees = _make(2, n)
    acc = torch.zeros((n, 3), device="cuda"); pot = torch.zeros(n, device="cuda")
    for t in trees:
        t.build(pos.cuda(), mass.cuda()); t.set_velocity(vel.cuda())
    force_local(trees, theta, eps, [(acc, pot), (None, None)])
    torch.cuda.synchronize()
    assert np.array_equal(acc.cpu().numpy(), r0["acc0"]) and np.array_equal(pot.cpu().numpy(), r0["pot0"])
    for _ in range(2):
        leapfrog_local(trees, dt)
    p = torch.empty((n, 3), device="cuda"); a = torch.empty((n, 3), device="cuda"); ph = torch.empty(n, device="cuda")
    trees[0].get_state(p, None, a, ph); torch.cuda.synchronize()
    assert np.array_equal(p.cpu().numpy(), r0["p"]) and np.array_equal(a.cpu().numpy(), r0["a"])
    ot = oracle.Tree(r0["p"], mass.numpy())
    oacc, opot, onpp, onpc = ot.force(theta, eps)
    assert np.array_equal(r0["counts"][:, 0], onpp) and np.array_equal(r0["counts"][:, 1], onpc)
    rel = np.linalg.norm(r0["a"].astype(np.float64) - oacc, axis=1) / np.linalg.norm(oacc, axis=1)
    assert rel.max() <= TOL
    _close(trees)


@pytest.mark.parametrize("n,world,dt", [(2000, 5, 0.5), (70000, 8, 0.05), (150, 8, 0.2), (30000, 3, 1e-3)])
def test_sharded_steps_cut_the_sort_by_key_range(n, world, dt):
    # A sharded step sorts by key range: context r sorts the particles whose new key falls between the splitters of the
    # previous order and stores the run into every context.  Large dt: particles move far, buckets become very uneven
    # (some empty); whatever the cut, every context must end with the oracle's order, tree and counts on the final
    # positions, bit-identical to a single context that sorted everything itself.
    theta, eps, steps = 0.4, 0.05, 3
    pos, vel, mass = plummer(n, 41)
    dpos, dvel, dmass = pos.cuda(), vel.cuda(), mass.cuda()
    one = Tree(device=0)
    one.build(dpos, dmass); one.set_velocity(dvel); one.force(theta, eps)
    trees = _make(world, n)
    for t in trees:
        t.build(dpos, dmass); t.set_velocity(dvel)
    force_local(trees, theta, eps)
    for _ in range(steps):
        one.leapfrog(dt)
        leapfrog_local(trees, dt)
    torch.cuda.synchronize()

    def state(t):
        p = torch.empty((n, 3), device="cuda"); v = torch.empty((n, 3), device="cuda")
        a = torch.empty((n, 3), device="cuda"); ph = torch.empty(n, device="cuda")
        t.get_state(p, v, a, ph); torch.cuda.synchronize()
        return p.cpu().numpy(), v.cpu().numpy(), a.cpu().numpy(), ph.cpu().numpy()

    p1, v1, a1, ph1 = state(one)
    p0, v0, a0, ph0 = state(trees[0])
    # (the single context's task list differs, so a few partial sums are ordered differently: close, not identical)
    assert np.abs(p0 - p1).max() <= 1e-5 * np.abs(p1).max()
    ot = oracle.Tree(p0, mass.numpy())
    key, order, skey = ot.keys()
    oacc, opot, onpp, onpc = ot.force(theta, eps)
    for t in trees:
        p, v, a, ph = state(t)
        assert np.array_equal(p, p0) and np.array_equal(v, v0)        # all contexts hold the same bits
        assert np.array_equal(t.debug("order"), order)
        assert np.array_equal(t.debug("sorted_keys"), skey)
        assert np.array_equal(t.debug("cells"), ot.cells())
        assert np.array_equal(t.debug("moments"), ot.moments())
        cnt = t.debug("counts")
        assert np.array_equal(cnt[:, 0], onpp) and np.array_equal(cnt[:, 1], onpc)
        rel = np.linalg.norm(a.astype(np.float64) - oacc, axis=1) / np.linalg.norm(oacc, axis=1)
        assert rel.max() <= TOL
    one.close()
    _close(trees)
