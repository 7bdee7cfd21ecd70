"""GPU parity of the error-targeted acceptance criterion (tree_set_mac_relative) against the oracle's
option "relative": with the SAME per-particle |a| given to both sides, per-group interaction counts are bit-exact and
forces agree to 1e-5; the library's own bookkeeping (|a| of its last pass, carried through tree_leapfrog) gives the same
lists as handing those values in; the criterion buys the canonical median error with fewer interactions."""
import numpy as np
import pytest
import torch

import oracle
from nbody_inputs import plummer, milky_way
from paper_1412_0659_b200 import Tree, TreeError

pytestmark = pytest.mark.gpu


def _amag_like_the_kernel(a32):
    """|a| as amag_acc_kernel forms it: sqrt(fma(az, az, fma(ay, ay, ax * ax))), FP32, one rounding each (long double holds
    the exact products and sums of FP32 operands here up to a 2^-40 chance of a double rounding)."""
    a = a32.astype(np.longdouble)
    x = (a[:, 0] * a[:, 0]).astype(np.float32).astype(np.longdouble)
    y = (a[:, 1] * a[:, 1] + x).astype(np.float32).astype(np.longdouble)
    z = (a[:, 2] * a[:, 2] + y).astype(np.float32)
    return np.sqrt(z)  # IEEE sqrt of an FP32 value in FP32


@pytest.mark.parametrize("model,n,seed,alpha,floor,leaf,group", [
    ("plummer", 16384, 1001, 1e-3, 1.0, 16, 64),
    ("mw", 100000 + 13, 3, 3e-4, 1.0, 16, 64),
    ("mw", 40000, 5, 3e-3, 0.7, 16, 64),
    ("plummer", 5000, 7, 1e-3, 1.0, 8, 32),
    ("mw", 30000, 9, 1e-3, 1.0, 16, 128),
    ("plummer", 3000, 11, 0.0, 1.0, 16, 64),
])
def test_relative_parity_with_the_same_accelerations_on_both_sides(model, n, seed, alpha, floor, leaf, group):
    eps = 0.01
    pos, _, mass = (plummer if model == "plummer" else milky_way)(n, seed, with_vel=False)
    ot = oracle.Tree(pos.numpy(), mass.numpy(), leaf_size=leaf, group_size=group)
    a0, _, pp0, pc0 = ot.force(0.4, eps)                           # the oracle's own canonical pass provides |a|
    amag = np.linalg.norm(a0, axis=1).astype(np.float32)
    ot.set_mac_relative(alpha, amag)
    oacc, opot, onpp, onpc = ot.force(floor, eps)
    t = Tree(device=0, leaf_size=leaf, group_size=group)
    acc = torch.empty((n, 3), device="cuda"); pot = torch.empty(n, device="cuda")
    t.build(pos.cuda(), mass.cuda())
    t.set_mac_relative(alpha, torch.from_numpy(amag).cuda())
    t.force(floor, eps, acc, pot)
    torch.cuda.synchronize()
    cnt = t.debug("counts")
    assert np.array_equal(cnt[:, 0], onpp) and np.array_equal(cnt[:, 1], onpc)
    if alpha > 0:
        assert (13.0 * onpp + 32.0 * onpc).sum() > 0 and not np.array_equal(onpc, pc0)   # the condition really decided
    a = acc.cpu().numpy().astype(np.float64); p = pot.cpu().numpy().astype(np.float64)
    assert (np.linalg.norm(a - oacc, axis=1) / np.linalg.norm(oacc, axis=1)).max() <= 1e-5
    assert (np.abs(p - opot) / np.abs(opot)).max() <= 1e-5
    # switched off again: the canonical lists, no rebuild needed
    t.set_mac("geometric")
    t.force(0.4, eps)
    cnt = t.debug("counts")
    assert np.array_equal(cnt[:, 0], pp0) and np.array_equal(cnt[:, 1], pc0)
    t.close()


def test_own_accelerations_travel_with_the_particles_through_leapfrog_steps():
    n, alpha, floor, eps, dt = 60000, 1e-3, 1.0, 0.01, 0.002
    pos, vel, mass = milky_way(n, 21)
    t = Tree(device=0)
    t.build(pos.cuda(), mass.cuda()); t.set_velocity(vel.cuda())
    t.force(0.4, eps)                      # no accelerations yet: the geometric criterion
    t.set_mac_relative(alpha)              # from here on scaled by the last pass
    t.force(floor, eps)
    for _ in range(2):
        t.leapfrog(dt)
    a_prev = torch.empty((n, 3), device="cuda")
    t.get_state(None, None, a_prev, None); torch.cuda.synchronize()
    amag = _amag_like_the_kernel(a_prev.cpu().numpy())
    t.leapfrog(dt)                         # this step's pass is scaled by |a_prev|, gathered into the new slot order
    p = torch.empty((n, 3), device="cuda"); a = torch.empty((n, 3), device="cuda")
    t.get_state(p, None, a, None); torch.cuda.synchronize()
    cnt = t.debug("counts")
    # the same pass with the values handed in: a second context built on the step's positions ...
    t2 = Tree(device=0)
    t2.build(p, mass.cuda())
    t2.set_mac_relative(alpha, torch.from_numpy(amag).cuda())
    t2.force(floor, eps)
    assert np.array_equal(t2.debug("counts"), cnt)
    t2.close()
    # ... and the oracle on the same input
    ot = oracle.Tree(p.cpu().numpy(), mass.numpy())
    ot.set_mac_relative(alpha, amag)
    oacc, _, onpp, onpc = ot.force(floor, eps)
    assert np.array_equal(cnt[:, 0], onpp) and np.array_equal(cnt[:, 1], onpc)
    rel = np.linalg.norm(a.cpu().numpy().astype(np.float64) - oacc, axis=1) / np.linalg.norm(oacc, axis=1)
    assert rel.max() <= 1e-5
    t.close()


def test_relative_criterion_buys_the_canonical_error_with_fewer_interactions():
    n, eps = 400000, 0.01
    pos, _, mass = milky_way(n, 33, with_vel=False)
    idx = torch.from_numpy(np.sort(np.random.default_rng(2001).choice(n, 8192, replace=False)).astype(np.int64)).cuda()
    t = Tree(device=0)
    acc = torch.empty((n, 3), device="cuda")
    t.build(pos.cuda(), mass.cuda())
    dacc = torch.empty((idx.numel(), 3), dtype=torch.float64, device="cuda")
    dpot = torch.empty(idx.numel(), dtype=torch.float64, device="cuda")
    t.direct(idx, eps, dacc, dpot)
    dn = dacc.norm(dim=1)

    def err():
        e = ((acc[idx].double() - dacc).norm(dim=1) / dn).cpu().numpy()
        _, pp, pc = t.stats()
        return np.median(e), np.percentile(e, 99), 13.0 * pp + 32.0 * pc
    t.force(0.4, eps, acc)
    m0, p0, c0 = err()
    t.set_mac_relative(3e-4)
    t.force(1.0, eps, acc)
    m1, p1, c1 = err()
    assert m1 <= m0 and p1 < p0 and c1 < 0.75 * c0, (m0, p0, m1, p1, c1 / c0)
    t.close()


def test_relative_criterion_argument_and_order_errors():
    pos, _, mass = plummer(2000, 3, with_vel=False)
    t = Tree(device=0)
    with pytest.raises(TreeError):
        t.set_mac_relative(-1.0)
    with pytest.raises(TreeError):                       # accelerations handed in before there is a slot order to put them in
        t.set_mac_relative(1e-3, torch.ones(2000, device="cuda"))
    t.set_mac("bmax")
    with pytest.raises(TreeError) as e:                  # the floor is the geometric criterion
        t.set_mac_relative(1e-3)
    assert e.value.code == -4
    t.set_mac("geometric")
    t.set_mac_relative(1e-3)                             # before any build: allowed, takes effect once a pass has run
    t.build(pos.cuda(), mass.cuda()); t.force(0.4, 0.01)
    c_geo = t.debug("counts").copy()
    t.force(1.0, 0.01)
    assert not np.array_equal(t.debug("counts"), c_geo)
    t.close()


def test_relative_criterion_on_sharded_contexts_equals_one_context():
    # every rank holds the complete results of every pass, so all ranks derive the same group scales: a sharded run in this
    # mode must reproduce the single context's lists and forces bit for bit, through force passes and leapfrog steps
    from paper_1412_0659_b200.sharded import connect_local, force_local, leapfrog_local
    n, alpha, eps, dt = 50000, 1e-3, 0.01, 0.002
    pos, vel, mass = milky_way(n, 17)
    dpos, dvel, dmass = pos.cuda(), vel.cuda(), mass.cuda()

    def run(world):
        trees = [Tree(device=0) for _ in range(world)]
        if world > 1:
            for t in trees:
                t.reserve(n)
            connect_local(trees)
        for t in trees:
            t.build(dpos, dmass); t.set_velocity(dvel)
        force_local(trees, 0.4, eps)
        for t in trees:
            t.set_mac_relative(alpha)
        force_local(trees, 1.0, eps)
        for _ in range(3):
            leapfrog_local(trees, dt)
        torch.cuda.synchronize()
        res = []
        for t in trees:
            p = torch.empty((n, 3), device="cuda"); a = torch.empty((n, 3), device="cuda")
            t.get_state(p, None, a, None); torch.cuda.synchronize()
            res.append((p.cpu(), a.cpu(), t.debug("counts").copy()))
            t.close()
        return res
    one = run(1)[0]
    for world in (2, 5):
        for p, a, c in run(world):
            assert torch.equal(p, one[0]) and torch.equal(a, one[1]) and np.array_equal(c, one[2])


def test_energy_drift_with_the_relative_criterion_is_no_worse_than_with_the_canonical_one():
    n, eps, dt, steps = 100000, 0.01, 0.001, 24
    pos, vel, mass = milky_way(n, 41)

    def drift(relative):
        t = Tree(device=0)
        t.build(pos.cuda(), mass.cuda()); t.set_velocity(vel.cuda()); t.force(0.4, eps)
        if relative:
            t.set_mac_relative(3e-4); t.force(1.0, eps)
        k0, p0 = t.energy()
        for _ in range(steps):
            t.leapfrog(dt)
        k1, p1 = t.energy()
        t.close()
        return abs((k1 + p1) - (k0 + p0)) / abs(k0 + p0)
    d_geo, d_rel = drift(False), drift(True)
    assert d_rel < max(3.0 * d_geo, 1e-6), (d_geo, d_rel)


def test_random_configurations_with_the_relative_criterion_against_oracle():
    """Seeded sweep: size, model, leaf and group size, alpha (0 and huge included), the geometric floor, eps, 1-3 sharded
    contexts, and the per-particle |a| either of the oracle's canonical pass or log-uniform random numbers (the scale is an
    input: any positive array must give the same lists on both sides)."""
    from paper_1412_0659_b200.sharded import connect_local, force_local
    import os
    rng = np.random.default_rng(20141207)
    for _ in range(int(os.environ.get("BH_FUZZ_CONFIGS", "24"))):  # a longer sweep of the same sequence: BH_FUZZ_CONFIGS=1000
        n = int(rng.choice([rng.integers(2, 200), rng.integers(200, 5000), rng.integers(5000, 30000)]))
        model = str(rng.choice(["plummer", "mw"])) if n >= 100 else "plummer"
        leaf = int(rng.choice([1, 8, 16, 32])); group = int(rng.choice([32, 64, 64, 128]))
        alpha = float(rng.choice([0.0 if n < 3000 else 1e-4, 1e-4, 1e-3, 1e-2, 1e30]))
        floor = float(rng.choice([0.5, 1.0, 1.0, 1.5])); eps = float(rng.choice([0.002, 0.01, 0.05]))
        world = int(rng.choice([1, 1, 2, 3])); seed = int(rng.integers(1, 10**6))
        pos, _, mass = (plummer if model == "plummer" else milky_way)(n, seed, with_vel=False)
        tag = f"n={n} {model} leaf={leaf} group={group} alpha={alpha} floor={floor} eps={eps} world={world} seed={seed}"
        ot = oracle.Tree(pos.numpy(), mass.numpy(), leaf_size=leaf, group_size=group)
        if rng.random() < 0.5:
            amag = np.linalg.norm(ot.force(0.4, eps)[0], axis=1).astype(np.float32)
        else:
            amag = (10.0 ** rng.uniform(-6, 3, n)).astype(np.float32)
        ot.set_mac_relative(alpha, amag)
        oacc, opot, onpp, onpc = ot.force(floor, eps)
        trees = [Tree(device=0, leaf_size=leaf, group_size=group) for _ in range(world)]
        for t in trees:
            t.reserve(n)
        if world > 1:
            connect_local(trees)
        damag = torch.from_numpy(amag).cuda()
        outs = [(torch.zeros((n, 3), device="cuda"), torch.zeros(n, device="cuda")) for _ in range(world)]
        for t in trees:
            t.build(pos.cuda(), mass.cuda()); t.set_mac_relative(alpha, damag)
        force_local(trees, floor, eps, outs)
        torch.cuda.synchronize()
        for t, (acc, pot) in zip(trees, outs):
            cnt = t.debug("counts")
            assert np.array_equal(cnt[:, 0], onpp) and np.array_equal(cnt[:, 1], onpc), tag
            a = acc.cpu().numpy().astype(np.float64); p = pot.cpu().numpy().astype(np.float64)
            relv = np.linalg.norm(a - oacc, axis=1) / np.linalg.norm(oacc, axis=1)
            i = int(relv.argmax())
            A = ot.abs_sum(floor, eps, [i])[0]
            assert relv.max() <= 1e-5 or np.linalg.norm(a[i] - oacc[i]) <= 2.5e-7 * A, (tag, relv.max())
            assert (np.abs(p - opot) / np.abs(opot)).max() <= 1e-5, tag
            t.close()


def test_switching_the_relative_criterion_off_and_on_again_starts_from_the_last_pass():
    # while it is off, steps do not carry |a| along; switching it on again must scale the next pass by the last pass's
    # accelerations in the CURRENT slot order, exactly as if those values were handed in
    n, alpha, eps, dt = 30000, 1e-3, 0.01, 0.002
    pos, vel, mass = milky_way(n, 23)
    t = Tree(device=0)
    t.build(pos.cuda(), mass.cuda()); t.set_velocity(vel.cuda())
    t.force(0.4, eps); t.set_mac_relative(alpha); t.force(1.0, eps); t.leapfrog(dt)
    t.set_mac("geometric")
    t.force(0.4, eps)
    for _ in range(2):
        t.leapfrog(dt)                      # canonical steps: the order changes, |a| is not gathered
    p = torch.empty((n, 3), device="cuda"); a = torch.empty((n, 3), device="cuda")
    t.get_state(p, None, a, None); torch.cuda.synchronize()
    t.set_mac_relative(alpha)               # NULL: |a| of the last (canonical) pass
    t.force(1.0, eps)
    cnt = t.debug("counts")
    t2 = Tree(device=0)
    t2.build(p, mass.cuda())
    t2.set_mac_relative(alpha, torch.from_numpy(_amag_like_the_kernel(a.cpu().numpy())).cuda())
    t2.force(1.0, eps)
    assert np.array_equal(t2.debug("counts"), cnt)
    t.close(); t2.close()


def test_relative_parity_at_bench_size_config3_sampled_groups():
    # BASELINE config 3 (Milky-Way-shaped, N = 8,388,608, eps = 0.01), the launch configuration bench.py times for it:
    # counts and forces against the oracle's option on every 509th group, with a smooth synthetic |a| as the common input
    # (enclosed mass of the three components over r^2 + 1: the scale is an input, any positive array will do)
    from nbody_inputs import config
    cfg, pos, vel, mass = config(2, with_vel=False)
    n, eps, alpha = cfg["n"], cfg["eps"], 3e-4
    r = pos.double().norm(dim=1).numpy()
    menc = 80.0 * np.minimum(r / 200.0, 1.0) + 5.0 * (1.0 - np.exp(-r / 2.5)) + 1.0 * (r / (r + 0.7)) ** 2
    amag = (menc / (r * r + 1.0)).astype(np.float32)
    t = Tree(device=0)
    acc = torch.empty((n, 3), device="cuda"); pot = torch.empty(n, device="cuda")
    t.build(pos.cuda(), mass.cuda())
    t.set_mac_relative(alpha, torch.from_numpy(amag).cuda())
    t.force(1.0, eps, acc, pot)
    torch.cuda.synchronize()
    ot = oracle.Tree(pos.numpy(), mass.numpy())
    order = ot.keys()[1]
    ot.set_mac_relative(alpha, amag)
    stride = 509
    oacc, opot, onpp, onpc = ot.force(1.0, eps, g0=3, stride=stride)
    gsel = np.arange(3, ot.n_groups, stride)
    cnt = t.debug("counts")
    assert np.array_equal(cnt[gsel, 0], onpp[gsel]) and np.array_equal(cnt[gsel, 1], onpc[gsel])
    sel = np.concatenate([order[64 * g: 64 * g + 64] for g in gsel])
    a = acc.cpu().numpy().astype(np.float64)[sel]; p = pot.cpu().numpy().astype(np.float64)[sel]
    assert (np.linalg.norm(a - oacc[sel], axis=1) / np.linalg.norm(oacc[sel], axis=1)).max() <= 1e-5
    assert (np.abs(p - opot[sel]) / np.abs(opot[sel])).max() <= 1e-5
    ms, pp, pc = t.stats()
    assert 2000 < (pp + pc) / n < 6000          # the condition is at work: the canonical theta = 1 lists are ~1500 long
    t.close()
