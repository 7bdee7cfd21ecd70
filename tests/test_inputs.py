"""Seeded input generators: determinism, index-addressability, shapes of the two models."""
import math

import numpy as np
import torch

from nbody_inputs import plummer, milky_way, uniform01, subsample_indices, config, CONFIGS
from nbody_inputs.generators import mw_counts


def test_uniform_is_counter_based():
    idx = torch.arange(1000, dtype=torch.int64)
    a = uniform01(5, idx, 2)
    b = torch.cat([uniform01(5, idx[:300], 2), uniform01(5, idx[300:], 2)])
    assert torch.equal(a, b)
    assert not torch.equal(a, uniform01(6, idx, 2)) and not torch.equal(a, uniform01(5, idx, 3))
    assert 0.0 < float(a.min()) and float(a.max()) < 1.0
    u = uniform01(9, torch.arange(200000, dtype=torch.int64), 0)
    assert abs(float(u.mean()) - 0.5) < 5e-3 and abs(float(u.var()) - 1 / 12) < 2e-3


def test_plummer_shape():
    pos, vel, m = plummer(20000, 42)
    assert pos.dtype == torch.float32 and pos.shape == (20000, 3) and vel.shape == (20000, 3)
    assert torch.equal(pos, plummer(20000, 42)[0])
    assert torch.equal(pos[:100], plummer(100, 42)[0])  # any particle can be generated on its own
    r = pos.double().norm(dim=1)
    assert abs(float(r.median()) - (0.4995 ** (-2 / 3) - 1) ** -0.5) < 0.05
    assert float(r.max()) < 38.8
    ke = 0.5 * float((m.double() * (vel.double() ** 2).sum(1)).sum())
    assert abs(ke - 3 * math.pi / 64) < 0.01  # virial: T = 3 pi / 64 for G = M = a = 1
    assert abs(float(m.double().sum()) - 1.0) < 1e-6
    assert len(np.unique(pos.numpy(), axis=0)) == 20000  # no coincident particles (S2)


def test_milky_way_shape():
    n = 60000
    pos, vel, m = milky_way(n, 43)
    nd, nb, nh = mw_counts(n)
    assert (nd, nb, nh) == (10000, 5000, 45000)
    md, mb, mh = (float(m[:nd].double().sum()), float(m[nd:nd + nb].double().sum()), float(m[nd + nb:].double().sum()))
    assert abs(md - 5) < 1e-4 and abs(mb - 1) < 1e-4 and abs(mh - 80) < 1e-3
    R = pos[:nd, :2].double().norm(dim=1)
    assert float(R.max()) <= 25.0 and abs(float(pos[:nd, 2].abs().median()) - 0.3 * math.atanh(0.5)) < 0.02
    rb = pos[nd:nd + nb].double().norm(dim=1)
    assert float(rb.max()) <= 10.0 + 1e-4 and abs(float(rb.median()) - 0.7 * math.sqrt(0.5 * (10 / 10.7) ** 2) / (1 - math.sqrt(0.5 * (10 / 10.7) ** 2))) < 0.1
    rh = pos[nd + nb:].double().norm(dim=1)
    assert float(rh.max()) <= 200.0 + 1e-3 and 40 < float(rh.median()) < 90
    assert bool(torch.isfinite(pos).all()) and bool(torch.isfinite(vel).all())
    assert len(np.unique(pos.numpy(), axis=0)) == n


def test_subsample_and_configs():
    s = subsample_indices(1000, 64)
    assert len(s) == 64 and len(torch.unique(s)) == 64 and bool((s[1:] > s[:-1]).all())
    assert torch.equal(s, subsample_indices(1000, 64))
    assert [CONFIGS[k]["n"] for k in range(5)] == [16384, 1048576, 8388608, 134217728, 33554432]
    cfg, pos, vel, m = config(0)
    assert cfg["eps"] == 0.01 and cfg["theta"] == 0.4 and pos.shape == (16384, 3)


def test_clumpy_disk_moves_only_disk_particles_and_is_seeded():
    import torch
    from nbody_inputs import milky_way, milky_way_clumpy
    from nbody_inputs.generators import mw_counts
    n = 48000
    p1, m1 = milky_way_clumpy(n, 9)
    p2, m2 = milky_way_clumpy(n, 9)
    q, _, mq = milky_way(n, 9, with_vel=False)
    assert torch.equal(p1, p2) and torch.equal(m1, m2) and torch.equal(m1, mq)
    nd, nb, nh = mw_counts(n)
    moved = (p1 != q).any(dim=1)
    assert int(moved.sum()) == int(nd * 0.2) and not bool(moved[int(nd * 0.2):].any())
    assert bool(torch.isfinite(p1).all()) and torch.unique(p1, dim=0).shape[0] == n
    # the clumps are compact: moved particles sit within a few scale radii of an unmoved disk particle
    d = torch.cdist(p1[moved][:200].double(), q[int(nd * 0.2):nd].double()).min(dim=1).values
    assert float(d.median()) < 0.1
