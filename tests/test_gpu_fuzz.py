"""Seeded random-configuration parity sweep (GPU): particle count, model, leaf and group size, theta, eps, planted far
outliers, 1-8 sharded contexts and 0-3 leapfrog steps are drawn at random; every configuration must reproduce the oracle's
sorted order, tree topology, moments and per-group interaction counts bit for bit and its forces within 1e-5 on the
positions of the last pass.  (DESIGN.md §5 "Accumulation" reports a 3000-configuration run of the same sweep.)"""
import numpy as np
import pytest
import torch

import oracle
from nbody_inputs import plummer, milky_way
from paper_1412_0659_b200 import Tree
from paper_1412_0659_b200.sharded import connect_local, force_local, leapfrog_local

pytestmark = pytest.mark.gpu


def _one(rng):
    n = int(rng.choice([rng.integers(1, 200), rng.integers(200, 5000), rng.integers(5000, 40000)]))
    model = str(rng.choice(["plummer", "mw"])) if n >= 100 else "plummer"
    leaf = int(rng.choice([1, 4, 8, 16, 32])); group = int(rng.choice([32, 64, 64, 128]))
    theta = float(rng.choice([0.0 if n < 3000 else 0.3, 0.3, 0.4, 0.4, 0.6, 0.9])); eps = float(rng.choice([0.002, 0.01, 0.05]))
    world = int(rng.choice([1, 1, 2, 3, 5, 8])); steps = int(rng.choice([0, 0, 1, 3]))
    seed = int(rng.integers(1, 10**6))
    pos, vel, mass = (plummer if model == "plummer" else milky_way)(n, seed)
    if rng.random() < 0.3 and n > 500:  # a few particles far from their Peano-Hilbert neighbours
        k = max(1, n // 997)
        idx = torch.from_numpy(rng.choice(n, k, replace=False))
        pos[idx] = torch.from_numpy(rng.normal(size=(k, 3)).astype(np.float32)) * 50
    tag = f"n={n} {model} leaf={leaf} group={group} theta={theta} eps={eps} world={world} steps={steps} seed={seed}"
    trees = [Tree(device=0, leaf_size=leaf, group_size=group) for _ in range(world)]
    for t in trees:
        t.reserve(n)
    if world > 1:
        connect_local(trees)
    for t in trees:
        t.build(pos.cuda(), mass.cuda()); t.set_velocity(vel.cuda())
    if world > 1:
        force_local(trees, theta, eps)
        for _ in range(steps):
            leapfrog_local(trees, 1e-3)
    else:
        trees[0].force(theta, eps)
        for _ in range(steps):
            trees[0].leapfrog(1e-3)
    torch.cuda.synchronize()
    t = trees[-1]
    p = torch.empty((n, 3), device="cuda"); a = torch.empty((n, 3), device="cuda"); ph = torch.empty(n, device="cuda")
    t.get_state(p, None, a, ph)
    torch.cuda.synchronize()
    ot = oracle.Tree(p.cpu().numpy(), mass.numpy(), leaf_size=leaf, group_size=group)
    assert np.array_equal(t.debug("order"), ot.keys()[1]), tag
    assert np.array_equal(t.debug("cells"), ot.cells()), tag
    assert np.array_equal(t.debug("moments"), ot.moments()), tag
    oacc, opot, onpp, onpc = ot.force(theta, eps)
    cnt = t.debug("counts")
    assert np.array_equal(cnt[:, 0], onpp) and np.array_equal(cnt[:, 1], onpc), tag
    if n > 1:
        an = a.cpu().numpy().astype(np.float64); pn = ph.cpu().numpy().astype(np.float64)
        rel = (np.linalg.norm(an - oacc, axis=1) / np.linalg.norm(oacc, axis=1)).max()
        prel = (np.abs(pn - opot) / np.abs(opot)).max()
        assert rel <= 1e-5 and prel <= 1e-5, (tag, rel, prel)
    for t in trees:
        t.close()


def test_random_configurations_against_oracle():
    rng = np.random.default_rng(20141206)
    for _ in range(48):
        _one(rng)
