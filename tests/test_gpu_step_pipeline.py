"""GPU tests of the step pipeline of tree_leapfrog: the state
stays in slot order between steps, the sort's payload is the previous slot, ties are re-ranked by caller index, the
rebuild does not wait for the host (cell arrays used up to a bound the device checks), the closing half kick runs in
the walk's epilogue.  What must hold is what held before: everything equals the oracle on the step's positions."""
import numpy as np
import pytest
import torch

import oracle
from nbody_inputs import plummer, milky_way
from paper_1412_0659_b200 import Tree, TreeError

pytestmark = pytest.mark.gpu


def _state(t, n):
    p = torch.empty((n, 3), device="cuda"); v = torch.empty((n, 3), device="cuda")
    a = torch.empty((n, 3), device="cuda"); ph = torch.empty(n, device="cuda")
    t.get_state(p, v, a, ph)
    torch.cuda.synchronize()
    return p.cpu().numpy(), v.cpu().numpy(), a.cpu().numpy(), ph.cpu().numpy()


def test_ties_formed_by_the_drift_are_ordered_by_caller_index():
    # Positions quantised far coarser than the key grid: a box of 2e-6 around 1.0, where FP32 has ~17 values per axis,
    # so thousands of particles share finest grid cells and ties form and break with every drift.  S10: equal keys are
    # ordered by CALLER index, although the sort inside tree_leapfrog carries the previous slot.
    n, eps, theta, dt = 6000, 1e-6, 0.4, 1.0
    rng = np.random.default_rng(3)
    pos = torch.from_numpy((1.0 + rng.random((n, 3)) * 2e-6).astype(np.float32))
    vel = torch.from_numpy((rng.normal(size=(n, 3)) * 2e-7).astype(np.float32))
    mass = torch.full((n,), 1e-12)  # negligible forces: the drift is the velocities'
    t = Tree(device=0)
    t.build(pos.cuda(), mass.cuda()); t.set_velocity(vel.cuda()); t.force(theta, eps)
    for step in range(4):
        t.leapfrog(dt)
        p, v, a, ph = _state(t, n)
        ot = oracle.Tree(p, mass.numpy())
        key, order, skey = ot.keys()
        ties = int((np.diff(skey) == 0).sum())
        assert ties > 100, ties  # the test does exercise ties
        assert np.array_equal(t.debug("order"), order), f"step {step}: sorted order differs ({ties} tied neighbours)"
        assert np.array_equal(t.debug("sorted_keys"), skey)
        assert np.array_equal(t.debug("cells"), ot.cells())
        assert np.array_equal(t.debug("moments"), ot.moments())
        assert np.array_equal(t.debug("sorted_pos")[:, :3], p[order])
    t.close()


def test_state_survives_many_steps_in_slot_order():
    # velocities, positions and caller indices travel together through 12 re-orderings: against the oracle's run
    n, dt, theta, eps, steps = 20000, 0.01, 0.4, 0.02, 12
    pos, vel, mass = plummer(n, 5)
    t = Tree(device=0)
    t.build(pos.cuda(), mass.cuda()); t.set_velocity(vel.cuda()); t.force(theta, eps)
    for _ in range(steps):
        t.leapfrog(dt)
    p, v, a, ph = _state(t, n)
    op, ov, oa, oph, en = oracle.leapfrog(pos.numpy(), vel.numpy(), mass.numpy(), dt, steps, theta, eps)
    assert np.abs(p - op).max() <= 2e-6 * np.abs(op).max()
    assert np.abs(v - ov).max() <= 2e-5 * np.abs(ov).max()
    ot = oracle.Tree(p, mass.numpy())
    assert np.array_equal(t.debug("order"), ot.keys()[1])
    oacc, opot, onpp, onpc = ot.force(theta, eps)
    cnt = t.debug("counts")
    assert np.array_equal(cnt[:, 0], onpp) and np.array_equal(cnt[:, 1], onpc)
    rel = np.linalg.norm(a.astype(np.float64) - oacc, axis=1) / np.linalg.norm(oacc, axis=1)
    assert rel.max() <= 1e-5
    # a new tree_build on the same context starts over (velocities must be set again)
    t.build(torch.from_numpy(p).cuda(), mass.cuda())
    with pytest.raises(TreeError) as e:
        t.leapfrog(dt)
    assert e.value.code == -4
    t.close()


def test_force_outputs_and_get_state_are_in_caller_order_after_steps():
    n, theta, eps = 5000 + 3, 0.4, 0.01
    pos, vel, mass = milky_way(n, 17)
    t = Tree(device=0)
    t.build(pos.cuda(), mass.cuda()); t.set_velocity(vel.cuda()); t.force(theta, eps)
    for _ in range(3):
        t.leapfrog(1e-3)
    p, v, a, ph = _state(t, n)
    acc = torch.empty((n, 3), device="cuda"); pot = torch.empty(n, device="cuda")
    t.force(theta, eps, acc, pot)  # same tree, same positions: the same force, now also to the caller's arrays
    torch.cuda.synchronize()
    assert np.array_equal(acc.cpu().numpy(), a) and np.array_equal(pot.cpu().numpy(), ph)
    ad, pd = oracle.direct(p, mass.numpy(), eps)
    rel = np.linalg.norm(a - ad, axis=1) / np.linalg.norm(ad, axis=1)
    assert np.median(rel) < 2e-3  # caller order is right: a permuted result would be off by O(1)
    t.close()


def test_asynchronous_rebuild_reports_cell_overflow_and_freezes_the_state():
    # 2500 clumps of 16 exactly coincident particles make a tree of ~3 k cells; one long drift with random velocities
    # blows every clump apart and the rebuilt tree needs ~4 x the cells allocated.  tree_leapfrog itself never waits for
    # the device: the step's kernels see the overflow flag and do nothing, and the next synchronising call reports
    # TREE_ERR_NOMEM once.  The state is frozen after that step's drift and a new tree_build continues from it.
    n, theta, eps = 40000, 0.4, 0.05
    rng = np.random.default_rng(11)
    centres = rng.normal(size=(n // 16, 3)).astype(np.float32)
    pos = torch.from_numpy(np.repeat(centres, 16, axis=0))
    vel = torch.from_numpy(rng.normal(size=(n, 3)).astype(np.float32))
    mass = torch.full((n,), 1.0 / n)
    t = Tree(device=0)
    t.build(pos.cuda(), mass.cuda()); t.set_velocity(vel.cuda()); t.force(theta, eps)
    cells0 = len(t.debug("cells"))
    p0, v0, a0, _ = _state(t, n)
    dt = 0.05
    t.leapfrog(dt)       # overflows on the device
    t.leapfrog(dt)       # enqueued behind it: must not move anything
    with pytest.raises(TreeError) as e:
        t.stats()
    assert e.value.code == -2, e.value
    p1 = torch.empty((n, 3), device="cuda"); v1 = torch.empty((n, 3), device="cuda")
    t.get_state(p1, v1, None, None)
    torch.cuda.synchronize()
    hdt = np.float32(0.5) * np.float32(dt)
    vh = (a0.astype(np.float64) * np.float64(hdt) + v0.astype(np.float64)).astype(np.float32)
    ph = (vh.astype(np.float64) * np.float64(np.float32(dt)) + p0.astype(np.float64)).astype(np.float32)
    assert np.array_equal(p1.cpu().numpy(), ph) and np.array_equal(v1.cpu().numpy(), vh)  # exactly one kick + drift
    with pytest.raises(TreeError) as e:
        t.leapfrog(dt)   # no tree any more
    assert e.value.code == -4
    t.build(p1, mass.cuda()); t.set_velocity(v1); t.force(theta, eps)
    assert len(t.debug("cells")) > 2 * cells0
    ot = oracle.Tree(p1.cpu().numpy(), mass.numpy())
    assert np.array_equal(t.debug("cells"), ot.cells())
    t.leapfrog(1e-3)
    t.stats()            # no error left over
    t.close()


def test_one_step_moves_few_particles_along_the_curve():
    # What the step pipeline relies on (and what it cannot use): after one step of BASELINE configs[4]'s dt most
    # particles keep their slot or move by a few slots, so the gather from the previous slot order is nearly sequential;
    # but almost every KEY changes in its low digits, so no pass of an LSD radix sort can be skipped.
    n, theta, eps, dt = 1 << 20, 0.4, 0.01, 0.0005
    pos, vel, mass = milky_way(n, 1005)
    t = Tree(device=0)
    t.build(pos.cuda(), mass.cuda()); t.set_velocity(vel.cuda()); t.force(theta, eps)
    t.leapfrog(dt)
    order0, key0 = t.debug("order").astype(np.int64), t.debug("sorted_keys")
    t.leapfrog(dt)
    order1, key1 = t.debug("order").astype(np.int64), t.debug("sorted_keys")
    slot0 = np.empty(n, np.int64); slot0[order0] = np.arange(n)
    slot1 = np.empty(n, np.int64); slot1[order1] = np.arange(n)
    disp = np.abs(slot1 - slot0)
    k0 = np.empty(n, np.uint64); k0[order0] = key0
    k1 = np.empty(n, np.uint64); k1[order1] = key1
    changed = k0 != k1
    low_byte_same = ((k0 ^ k1) & np.uint64(0xff)) == 0
    print(f"\nslots: unchanged {np.mean(disp == 0):.3f}, moved <= 32 {np.mean(disp <= 32):.4f}, <= 2048 {np.mean(disp <= 2048):.5f}, "
          f"max {disp.max()}; keys changed {changed.mean():.4f}, lowest byte unchanged {low_byte_same.mean():.4f}")
    assert np.mean(disp <= 32) > 0.97          # the gather reads within a cache line or two of where it writes
    assert changed.mean() > 0.9                # yet nearly every key differs: nothing for a radix pass to skip
    t.close()


def test_caller_order_results_from_the_walk_epilogue_equal_the_state_also_for_split_groups():
    # tree_force with caller arrays on one context writes them in the walk's epilogue (a11 fused): the arrays must hold exactly
    # what tree_get_state returns afterwards, also for groups whose walk was cut into parts (their results are written by the part
    # that combines the partial sums) and for acc-only / pot-only calls
    n, theta, eps = 200_000, 0.4, 0.01
    pos, _, mass = plummer(n, 91, with_vel=False)
    idx = torch.arange(0, n, 1500)   # a few particles far out: their runs of 64 have boxes over dense regions and are split
    d = torch.randn(len(idx), 3, generator=torch.Generator().manual_seed(6), dtype=torch.float64)
    pos[idx] = (25.0 * d / d.norm(dim=1, keepdim=True)).float()
    t = Tree(device=0)
    acc = torch.full((n, 3), float("nan"), device="cuda"); pot = torch.full((n,), float("nan"), device="cuda")
    t.build(pos.cuda(), mass.cuda())
    t.force(theta, eps, acc, pot)
    tr = t.debug("task_trace")
    assert ((tr[:, 3] >> 26) > 0).any()          # some groups were walked in parts
    a2 = torch.empty((n, 3), device="cuda"); p2 = torch.empty(n, device="cuda")
    t.get_state(None, None, a2, p2); torch.cuda.synchronize()
    assert torch.equal(acc, a2) and torch.equal(pot, p2)
    # acc only / pot only (a later pass is scheduled by the previous one's counts: other parts, other last bits, so every
    # pass is compared with its own state)
    acc.fill_(float("nan")); t.force(theta, eps, acc, None)
    t.get_state(None, None, a2, p2); torch.cuda.synchronize()
    assert torch.equal(acc, a2)
    pot.fill_(float("nan")); t.force(theta, eps, None, pot)
    t.get_state(None, None, a2, p2); torch.cuda.synchronize()
    assert torch.equal(pot, p2)
    t.close()
