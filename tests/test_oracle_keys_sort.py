"""Pins for the oracle's T1-T4 (bbox, grid, Peano-Hilbert key, stable sort). CPU only."""
import itertools
import os

import numpy as np
import pytest

import oracle
from nbody_inputs import plummer

GOLD = os.path.join(os.path.dirname(__file__), "golden", "hilbert_pins.txt")


def test_hilbert_golden_values():
    n = 0
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        bits, ix, iy, iz, key = (int(v) for v in line.split())
        assert oracle.hilbert_key(ix, iy, iz, bits) == key, line
        n += 1
    assert n >= 14


@pytest.mark.parametrize("bits", [1, 2, 3, 4])
def test_hilbert_bijection_adjacency_parent(bits):
    side = 1 << bits
    inv = {}
    for x, y, z in itertools.product(range(side), repeat=3):
        k = oracle.hilbert_key(x, y, z, bits)
        assert 0 <= k < side ** 3
        assert k not in inv  # injective => bijective onto [0, 8^bits)
        inv[k] = (x, y, z)
        if bits > 1:  # key >> 3 is the key of the parent cell at bits-1
            assert k >> 3 == oracle.hilbert_key(x >> 1, y >> 1, z >> 1, bits - 1)
    assert len(inv) == side ** 3
    for k in range(side ** 3 - 1):  # consecutive keys = face-adjacent cells
        a, b = inv[k], inv[k + 1]
        assert sum(abs(a[d] - b[d]) for d in range(3)) == 1


def test_hilbert_21bit_parent_and_locality():
    rng = np.random.default_rng(3)
    pts = rng.integers(0, 1 << 21, size=(200, 3))
    for x, y, z in pts:
        k = oracle.hilbert_key(x, y, z, 21)
        assert 0 <= k < 1 << 63
        for up in (1, 5, 13):
            assert k >> (3 * up) == oracle.hilbert_key(x >> up, y >> up, z >> up, 21 - up)


def test_grid_mapping_hand_checked():
    # lo = (0,0,0), hi = (1,1,3): ext = 3 -> side S = 4 (k = 2); centre (0.5,0.5,1.5);
    # origin = centre - 2 = (-1.5,-1.5,-0.5); scale = 2^21 / 4 = 2^19.
    pos = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 3]], np.float32)
    t = oracle.Tree(pos, np.ones(4, np.float32))
    lo, hi, org, k = t.grid()
    assert k == 2
    assert np.array_equal(lo, [0, 0, 0]) and np.array_equal(hi, [1, 1, 3])
    assert np.array_equal(org, np.array([-1.5, -1.5, -0.5], np.float32))
    key, order, skey = t.keys()
    sc = 1 << 19
    exp_idx = [(int(1.5 * sc), int(1.5 * sc), int(0.5 * sc)), (int(2.5 * sc), int(1.5 * sc), int(0.5 * sc)),
               (int(1.5 * sc), int(2.5 * sc), int(0.5 * sc)), (int(1.5 * sc), int(1.5 * sc), int(3.5 * sc))]
    for i, (ix, iy, iz) in enumerate(exp_idx):
        assert 0 <= min(ix, iy, iz) and max(ix, iy, iz) < 1 << 21
        assert int(key[i]) == oracle.hilbert_key(ix, iy, iz, 21)


def test_grid_power_of_two_side_and_bounds():
    for ext, k_exp in [(0.3, -1), (0.5, 0), (0.999, 0), (1.0, 1), (37.0, 6), (64.0, 7)]:
        pos = np.array([[0, 0, 0], [ext, 0.1 * ext, 0.2 * ext]], np.float32)
        t = oracle.Tree(pos, np.ones(2, np.float32))
        _, _, org, k = t.grid()
        assert k == k_exp, (ext, k)
        side = 2.0 ** k
        assert np.all(org <= pos.min(0)) and np.all(pos.max(0) < org + side)
    # all particles identical position: ext = 0 -> k = 0
    pos = np.ones((3, 3), np.float32)
    assert oracle.Tree(pos, np.ones(3, np.float32)).grid()[3] == 0


def test_sort_is_stable_permutation():
    pos, _, m = plummer(5000, 11, with_vel=False)
    pos = pos.numpy().copy()
    pos[100:140] = pos[7]  # coincident particles: equal keys, order must stay by index
    pos[4000:4010] = pos[7]
    t = oracle.Tree(pos, m.numpy())
    key, order, skey = t.keys()
    assert np.array_equal(np.sort(order), np.arange(5000, dtype=np.uint32))
    assert np.array_equal(skey, key[order])
    assert np.all(skey[1:] >= skey[:-1])
    same = skey[1:] == skey[:-1]
    assert same.sum() >= 49
    assert np.all(order[1:][same] > order[:-1][same])
    # sorted particle copy follows the permutation
    sp = t.sorted_particles()
    assert np.array_equal(sp[:, :3], pos[order]) and np.array_equal(sp[:, 3], m.numpy()[order])


def test_non_finite_input_is_an_error():
    pos = np.zeros((4, 3), np.float32)
    pos[2, 1] = np.nan
    with pytest.raises(ValueError):
        oracle.Tree(pos, np.ones(4, np.float32))
