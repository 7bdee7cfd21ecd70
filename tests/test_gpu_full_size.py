"""GPU parity at BASELINE.json's two largest configurations, in the launch configuration bench.py times:
configs[3] (Milky-Way-shaped, N = 134,217,728: the headline workload) and configs[4] (N = 33,554,432, 16
kick-drift-kick steps).  Integer and index work bit-exact on the FULL arrays (keys, order, cells, moments,
group boxes, opening radii); interaction counts bit-exact and forces within 1e-5 of the oracle's FP64 sum
on sampled groups (the oracle walks a group in ~1 ms: every group of 2 M would take half an hour)."""
import gc

import numpy as np
import pytest
import torch

import oracle
from nbody_inputs import config
from paper_1412_0659_b200 import Tree

pytestmark = pytest.mark.gpu

TOL = 1e-5  # north_star: max over particles, FP32 GPU tree vs the CPU tree


def _full_arrays_equal(t, ot):
    """Every array of the build, one at a time (the largest is 1.4 GB per side at 134 M)."""
    g = t.debug("grid")
    lo, hi, org, k = ot.grid()
    assert np.array_equal(g[:3], lo) and np.array_equal(g[3:6], hi) and np.array_equal(g[6:9], org) and g[9] == k
    key, order, skey = ot.keys()
    assert np.array_equal(t.debug("keys"), key), "PH keys differ"
    del key
    assert np.array_equal(t.debug("order"), order), "sorted order differs"
    assert np.array_equal(t.debug("sorted_keys"), skey), "sorted keys differ"
    del skey
    gc.collect()
    assert np.array_equal(t.debug("sorted_pos"), ot.sorted_particles()), "permuted particles differ"
    gc.collect()
    assert np.array_equal(t.debug("level_offsets")[-1], ot.n_cells)
    assert np.array_equal(t.debug("cells"), ot.cells()), "tree topology differs"
    gc.collect()
    assert np.array_equal(t.debug("moments"), ot.moments()), "multipole moments differ"
    gc.collect()
    gmin, gmax = ot.groups()
    gb = t.debug("group_boxes")
    assert np.array_equal(gb[:, :3], gmin) and np.array_equal(gb[:, 3:], gmax), "group boxes differ"
    return order


def _sampled_force_parity(t, ot, order, acc, pot, theta, eps, g0, stride):
    """Counts bit-exact and forces <= TOL on the groups g0, g0 + stride, ... (acc, pot: caller order, numpy f32)."""
    oacc, opot, onpp, onpc = ot.force(theta, eps, g0=g0, stride=stride)
    assert np.array_equal(t.debug("ropen2"), ot.ropen2()), "opening radii differ"
    gsel = np.arange(g0, ot.n_groups, stride)
    cnt = t.debug("counts")
    assert np.array_equal(cnt[gsel, 0], onpp[gsel]) and np.array_equal(cnt[gsel, 1], onpc[gsel]), "interaction counts differ"
    gs = ot.group_size
    sel = np.concatenate([order[gs * g: min(gs * g + gs, ot.n)] for g in gsel]).astype(np.int64)
    a = acc[sel].astype(np.float64); p = pot[sel].astype(np.float64)
    rel = np.linalg.norm(a - oacc[sel], axis=1) / np.linalg.norm(oacc[sel], axis=1)
    prel = np.abs(p - opot[sel]) / np.abs(opot[sel])
    assert rel.max() <= TOL, rel.max()
    assert prel.max() <= TOL, prel.max()
    return len(gsel), float(rel.max()), float(prel.max())


def test_config4_134m_full_arrays_and_sampled_forces():
    # BASELINE configs[3]: N = 134,217,728, eps = 0.005, theta = 0.4 -- bench.py's headline workload.  At this
    # size the scan runs 16 k blocks, the tree has ~32 M cells, the sort 65 k tiles with look-back chains.
    cfg, pos, vel, mass = config(3, device="cuda", with_vel=False)
    n = cfg["n"]
    t = Tree(device=0)
    acc = torch.empty((n, 3), device="cuda"); pot = torch.empty(n, device="cuda")
    t.build(pos, mass); t.force(cfg["theta"], cfg["eps"], acc, pot)
    torch.cuda.synchronize()
    ms, pp, pc = t.stats()  # raises if the walk's stack guard fired
    hpos, hmass = pos.cpu().numpy(), mass.cpu().numpy()
    hacc, hpot = acc.cpu().numpy(), pot.cpu().numpy()
    del pos, mass, acc, pot
    ot = oracle.Tree(hpos, hmass)
    order = _full_arrays_equal(t, ot)
    # every 4093rd group (a prime stride, so the sample drifts across tiles, blocks and the task list's regions)
    ng, amax, pmax = _sampled_force_parity(t, ot, order, hacc, hpot, cfg["theta"], cfg["eps"], g0=7, stride=4093)
    assert ng >= 512
    assert np.isfinite(hacc).all() and np.isfinite(hpot).all()
    print(f"config 4: {ot.n_cells} cells, {ng} groups checked, max rel acc {amax:.2e} pot {pmax:.2e}, "
          f"{pp / n:.0f} p-p + {pc / n:.0f} p-c per particle")
    t.close()


def test_config5_33m_16_leapfrog_steps_then_parity():
    # BASELINE configs[4]: N = 33,554,432, 16 kick-drift-kick steps of dt = 0.0005, each a full re-key, sort,
    # rebuild, moments and force pass scheduled by the previous step's counts.  The force of the LAST step must
    # be the oracle's force on the positions of that step: the oracle's tree is built on the final positions.
    cfg, pos, vel, mass = config(4, device="cuda")
    n, dt = cfg["n"], cfg["dt"]
    t = Tree(device=0)
    t.build(pos, mass); t.set_velocity(vel); t.force(cfg["theta"], cfg["eps"])
    e0 = sum(t.energy())
    for _ in range(cfg["steps"]):
        t.leapfrog(dt)
    e1 = sum(t.energy())
    p = torch.empty((n, 3), device="cuda"); a = torch.empty((n, 3), device="cuda"); ph = torch.empty(n, device="cuda")
    t.get_state(p, None, a, ph)
    torch.cuda.synchronize()
    ms, pp, pc = t.stats()
    hp, ha, hph, hmass = p.cpu().numpy(), a.cpu().numpy(), ph.cpu().numpy(), mass.cpu().numpy()
    assert not np.array_equal(hp, pos.cpu().numpy())  # the particles did move
    del pos, vel, mass, p, a, ph
    ot = oracle.Tree(hp, hmass)
    order = _full_arrays_equal(t, ot)
    ng, amax, pmax = _sampled_force_parity(t, ot, order, ha, hph, cfg["theta"], cfg["eps"], g0=3, stride=1021)
    assert ng >= 512
    drift = abs(e1 - e0) / abs(e0)
    assert drift < 1e-6, drift  # 16 steps of dt = 0.0005 (time unit 4.7 Myr); bench.py reports it beside the oracle's
    print(f"config 5: {ng} groups checked after 16 steps, max rel acc {amax:.2e} pot {pmax:.2e}, energy drift {drift:.2e}")
    t.close()
