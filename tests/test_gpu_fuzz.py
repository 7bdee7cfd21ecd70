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


def _one(rng, strict=True):
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
        relv = np.linalg.norm(an - oacc, axis=1) / np.linalg.norm(oacc, axis=1)
        rel = relv.max()
        prel = (np.abs(pn - opot) / np.abs(opot)).max()
        # the statement of DESIGN.md "Tolerance": |a_gpu - a_oracle| <= max(1e-5 |a_i|, 2.5e-7 A_i), A_i = sum of the
        # magnitudes of the terms of particle i's interaction list (the second term decides only where the sum cancels);
        # the committed 48 configurations (strict) meet both the plain 1e-5 bound and the A_i form for their worst particle
        i = int(relv.argmax())
        A = ot.abs_sum(theta, eps, [i])[0]
        err = np.linalg.norm(an[i] - oacc[i])
        assert prel <= 1e-5, (tag, prel)
        if strict:
            assert rel <= 1e-5, (tag, rel)
            assert err <= 2.5e-7 * A, (tag, i, err / A)
        else:
            assert rel <= 1e-5 or err <= 2.5e-7 * A, (tag, i, rel, err / A)
    for t in trees:
        t.close()


def test_random_configurations_against_oracle():
    import os
    rng = np.random.default_rng(20141206)
    for k in range(int(os.environ.get("BH_FUZZ_CONFIGS", "48"))):  # a longer sweep of the same sequence: BH_FUZZ_CONFIGS=3000
        _one(rng, strict=k < 48)


def _degenerate(rng, kind, n):
    if kind == "line":
        x = rng.random((n, 1)); p = np.concatenate([x, 0 * x + 0.25, 0 * x - 3.0], 1)
    elif kind == "plane":
        p = np.concatenate([rng.random((n, 2)), np.zeros((n, 1)) + 1.5], 1)
    elif kind == "lattice":
        k = int(np.ceil(n ** (1 / 3)))
        p = np.stack(np.meshgrid(*[np.arange(k)] * 3, indexing="ij"), -1).reshape(-1, 3)[:n].astype(np.float64) * 0.125
    elif kind == "dups":  # many exactly coincident particles: equal keys, leaves at the last level
        m = max(1, n // 40); p = rng.normal(size=(m, 3))[rng.integers(0, m, n)]
    elif kind == "clumps":
        c = rng.normal(size=(5, 3)) * 10
        p = c[rng.integers(0, 5, n)] + rng.normal(size=(n, 3)) * 10.0 ** rng.integers(-5, 0, (n, 1))
    elif kind == "huge":
        p = rng.normal(size=(n, 3)) * 1e4 + 3e5
    else:  # "tinybox": extent near the FP32 resolution of the coordinates
        p = 1.0 + rng.random((n, 3)) * 1e-5
    return torch.from_numpy(p.astype(np.float32))


def test_degenerate_geometries_against_oracle():
    """Lines, planes, lattices (tied keys), coincident particles, clumps over five decades, far-offset and
    resolution-limited boxes: keys, order, topology, moments and counts bit-exact, potentials within 1e-5.  The net
    acceleration cancels (exactly, by symmetry, or nearly) in several of these, so it is only checked to be finite and
    within 1e-3 of the largest acceleration in the set (a 20,000-configuration run of this sweep found no other deviation)."""
    rng = np.random.default_rng(7)
    kinds = ["line", "plane", "lattice", "dups", "clumps", "huge", "tinybox"]
    import os
    for it in range(int(os.environ.get("BH_FUZZ_DEGENERATE", "56"))):
        kind = kinds[it % len(kinds)]
        n = int(rng.choice([1, 2, 16, 17, 64, 65, 129, 1000, 4097, int(rng.integers(2, 20000))]))
        leaf = int(rng.choice([1, 8, 16, 32])); group = int(rng.choice([32, 64, 128]))
        theta = float(rng.choice([0.0 if n <= 4097 else 0.4, 0.4, 0.8, 1.5])); eps = float(rng.choice([0.01, 1e-3, 0.5]))
        pos = _degenerate(rng, kind, n)
        mass = torch.from_numpy((10.0 ** rng.uniform(-6, 0, n)).astype(np.float32)) if it % 2 else torch.full((n,), 1.0 / n)
        tag = f"{kind} n={n} leaf={leaf} group={group} theta={theta} eps={eps}"
        t = Tree(device=0, leaf_size=leaf, group_size=group)
        a = torch.empty((n, 3), device="cuda"); ph = torch.empty(n, device="cuda")
        t.build(pos.cuda(), mass.cuda()); t.force(theta, eps, a, ph)
        torch.cuda.synchronize()
        ot = oracle.Tree(pos.numpy(), mass.numpy(), leaf_size=leaf, group_size=group)
        assert np.array_equal(t.debug("keys"), ot.keys()[0]), tag
        assert np.array_equal(t.debug("order"), ot.keys()[1]), tag
        assert np.array_equal(t.debug("cells"), ot.cells()), tag
        assert np.array_equal(t.debug("moments"), ot.moments()), tag
        oacc, opot, onpp, onpc = ot.force(theta, eps)
        cnt = t.debug("counts")
        assert np.array_equal(cnt[:, 0], onpp) and np.array_equal(cnt[:, 1], onpc), tag
        an = a.cpu().numpy().astype(np.float64); pn = ph.cpu().numpy().astype(np.float64)
        assert np.isfinite(an).all() and np.isfinite(pn).all(), tag
        if n > 1:
            assert (np.abs(pn - opot) / np.abs(opot)).max() <= 1e-5, tag
            assert np.linalg.norm(an - oacc, axis=1).max() <= 1e-3 * np.linalg.norm(oacc, axis=1).max(), tag
        t.close()


def test_error_tail_report():
    """Random configurations for BH_TAIL_SECONDS (default 20 s; profiles/r2_tolerance_tail.md is a 300 s run with -s):
    the largest relative acceleration error of each, its cancellation factor kappa = A_i / |a_i| and its error in units
    of A_i.  Every worst particle must obey |err| <= max(1e-5 |a_i|, 2.5e-7 A_i)."""
    import os, time
    budget = float(os.environ.get("BH_TAIL_SECONDS", "20"))
    rng = np.random.default_rng(int(os.environ.get("BH_TAIL_SEED", "4242")))
    t0 = time.time(); res = []
    while time.time() - t0 < budget:
        n = int(rng.choice([rng.integers(200, 5000), rng.integers(5000, 40000), rng.integers(40000, 250000)]))
        model = str(rng.choice(["plummer", "mw"]))
        leaf = int(rng.choice([8, 16, 32]))
        theta = float(rng.choice([0.3, 0.4, 0.4, 0.6, 0.9])); eps = float(rng.choice([0.002, 0.01, 0.05]))
        seed = int(rng.integers(1, 10**6))
        pos, vel, mass = (plummer if model == "plummer" else milky_way)(n, seed)
        t = Tree(device=0, leaf_size=leaf, group_size=64)
        a = torch.empty((n, 3), device="cuda"); ph = torch.empty(n, device="cuda")
        t.build(pos.cuda(), mass.cuda()); t.force(theta, eps, a, ph); torch.cuda.synchronize()
        ot = oracle.Tree(pos.numpy(), mass.numpy(), leaf_size=leaf, group_size=64)
        oacc, opot, onpp, onpc = ot.force(theta, eps)
        an = a.cpu().numpy().astype(np.float64); pn = ph.cpu().numpy().astype(np.float64)
        rel = np.linalg.norm(an - oacc, axis=1) / np.linalg.norm(oacc, axis=1); prel = np.abs(pn - opot) / np.abs(opot)
        i = int(rel.argmax())
        A = ot.abs_sum(theta, eps, [i])[0]
        err = np.linalg.norm(an[i] - oacc[i])
        res.append((rel.max(), prel.max(), n, model, leaf, theta, eps, seed, A / np.linalg.norm(oacc[i]), err / A))
        assert err <= max(1e-5 * np.linalg.norm(oacc[i]), 2.5e-7 * A), res[-1]
        assert prel.max() <= 1e-5, res[-1]
        t.close()
    res.sort(reverse=True)
    above = sum(r[0] > 1e-5 for r in res)
    print(f"\n{len(res)} random configurations in {budget:.0f} s; max relative acceleration error above 1e-5 in {above}; "
          f"median of the maxima {np.median([r[0] for r in res]):.2e}; largest potential error {max(r[1] for r in res):.2e}")
    print("| max rel acc err | max rel pot err | N | model | leaf | theta | eps | seed | kappa = A_i / |a_i| | err / A_i |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    for r in res[:10]:
        print("| %.2e | %.2e | %d | %s | %d | %.1f | %g | %d | %.1f | %.2e |" % r)
    assert above <= max(1, len(res) // 200)
