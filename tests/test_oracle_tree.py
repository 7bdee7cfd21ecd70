"""Pins for the oracle's T5-T8 (octree, moments, groups). CPU only."""
import numpy as np
import pytest

import oracle
from nbody_inputs import plummer, milky_way


def _inputs(kind, n):
    if kind == "plummer":
        pos, _, m = plummer(n, 21, with_vel=False)
    elif kind == "mw":
        pos, _, m = milky_way(n, 22, with_vel=False)
    else:  # clumped: many coincident particles => level-21 leaves with more than 16 particles
        pos, _, m = plummer(n, 23, with_vel=False)
        pos = pos.clone()
        pos[: n // 8] = pos[0]
        pos[n // 8: n // 4] = pos[n // 8] + 1e-7
    return pos.numpy(), m.numpy()


def _python_tree(skey, leaf):
    """Independent builder: plain recursion on the sorted keys, then BFS renumbering."""
    nodes = []

    def rec(level, first, count):
        node = dict(level=level, first=first, count=count, kids=[])
        nodes.append(node)
        if count > leaf and level < 21:
            sh = 3 * (20 - level)
            dig = (skey[first:first + count] >> np.uint64(sh)) & np.uint64(7)
            cuts = np.flatnonzero(dig[1:] != dig[:-1]) + 1
            bounds = np.concatenate(([0], cuts, [count]))
            for a, b in zip(bounds[:-1], bounds[1:]):
                node["kids"].append(rec(level + 1, first + int(a), int(b - a)))
        return node

    root = rec(0, 0, len(skey))
    out, frontier = [], [root]
    while frontier:  # level by level, within a level in key order
        nxt = []
        for nd in frontier:
            nd["id"] = len(out)
            out.append(nd)
        for nd in frontier:
            nxt.extend(nd["kids"])
        frontier = nxt
    rec_arr = np.zeros((len(out), 5), np.int32)
    for nd in out:
        fc = nd["kids"][0]["id"] if nd["kids"] else -1
        rec_arr[nd["id"]] = (nd["level"], nd["first"], nd["count"], fc, len(nd["kids"]))
    return rec_arr


@pytest.mark.parametrize("kind,n", [("plummer", 4096), ("mw", 6000), ("clumped", 2048)])
def test_tree_invariants_and_independent_builder(kind, n):
    pos, m = _inputs(kind, n)
    t = oracle.Tree(pos, m)
    cells = t.cells()
    _, _, skey = t.keys()
    lvl, first, cnt, fc, nch = cells.T
    assert lvl[0] == 0 and first[0] == 0 and cnt[0] == n
    assert lvl.max() <= 21
    assert np.all(np.diff(lvl) >= 0)  # BFS: levels non-decreasing
    leaf = fc < 0
    # leaves tile [0, N) exactly once, in order
    lf = np.argsort(first[leaf], kind="stable")
    fs, cs = first[leaf][lf], cnt[leaf][lf]
    assert fs[0] == 0 and np.array_equal(fs[1:], (fs + cs)[:-1]) and fs[-1] + cs[-1] == n
    assert np.all((cnt[leaf] <= 16) | (lvl[leaf] == 21))
    assert np.all(cnt[~leaf] > 16) and np.all(lvl[~leaf] < 21)
    if kind == "clumped":
        assert np.any((cnt > 16) & leaf)  # exercises the level-21 rule
    for c in np.flatnonzero(~leaf):
        ch = np.arange(fc[c], fc[c] + nch[c])
        assert 1 <= nch[c] <= 8
        assert np.all(lvl[ch] == lvl[c] + 1)
        assert first[ch[0]] == first[c] and first[ch[-1]] + cnt[ch[-1]] == first[c] + cnt[c]
        assert np.array_equal(first[ch][1:], (first[ch] + cnt[ch])[:-1])
        sh = np.uint64(3 * (20 - lvl[c]))
        dig = [(int(skey[first[k]]) >> int(sh)) & 7 for k in ch]
        assert all(a < b for a, b in zip(dig[:-1], dig[1:]))  # distinct, key order
        for k in ch:  # all particles of a child share the digit and the parent's prefix
            ks = skey[first[k]: first[k] + cnt[k]] >> sh
            assert np.all(ks == ks[0])
    assert np.array_equal(cells, _python_tree(skey, 16))


def test_small_n_is_single_leaf_root():
    for n in (1, 2, 16):
        pos, _, m = plummer(n, 5, with_vel=False)
        t = oracle.Tree(pos.numpy(), m.numpy())
        assert t.n_cells == 1
        assert np.array_equal(t.cells()[0], [0, 0, n, -1, 0])
    pos, _, m = plummer(17, 5, with_vel=False)
    assert oracle.Tree(pos.numpy(), m.numpy()).n_cells > 1


@pytest.mark.parametrize("kind,n", [("plummer", 4096), ("mw", 6000)])
def test_moments_against_plain_definitions(kind, n):
    pos, m = _inputs(kind, n)
    t = oracle.Tree(pos, m)
    cells, mom = t.cells(), t.moments()
    sp = t.sorted_particles().astype(np.float64)
    _, _, org, k = t.grid()
    S = 2.0 ** k
    # every cell against the FP64 definition over its own particle range (S4: raw second
    # central moment, not traceless, not per unit mass)
    for c in range(t.n_cells):
        lv, f, cn, fc, nc = cells[c]
        x, w = sp[f:f + cn, :3], sp[f:f + cn, 3]
        M = w.sum()
        com = (w[:, None] * x).sum(0) / M
        d = x - com
        Q = np.einsum("k,ka,kb->ab", w, d, d)
        assert abs(mom[c, 0] - M) <= 1e-6 * M
        lc = S / 2 ** lv
        assert np.all(np.abs(mom[c, 1:4] - com) <= 2e-6 * max(lc, np.abs(com).max()))
        qref = np.array([Q[0, 0], Q[1, 1], Q[2, 2], Q[0, 1], Q[0, 2], Q[1, 2]])
        assert np.all(np.abs(mom[c, 4:10] - qref) <= 2e-5 * max(np.trace(Q), 1e-30)), c
        # positive semi-definite, trace >= 0
        Qm = np.array([[mom[c, 4], mom[c, 7], mom[c, 8]], [mom[c, 7], mom[c, 5], mom[c, 9]],
                       [mom[c, 8], mom[c, 9], mom[c, 6]]], np.float64)
        assert np.linalg.eigvalsh(Qm).min() >= -1e-6 * max(np.trace(Qm), 1e-30)
        # delta = |com - geometric centre| <= half diagonal; centre from the cell's key prefix
        assert mom[c, 10] <= (np.sqrt(3) / 2) * lc * (1 + 1e-6)
        q = np.floor((x[0] - org.astype(np.float64)) / lc)
        gcen = org + (q + 0.5) * lc
        assert abs(mom[c, 10] - np.linalg.norm(mom[c, 1:4].astype(np.float64) - gcen)) <= 1e-5 * lc
        if cn == 1:
            assert np.all(mom[c, 4:10] == 0) and np.all(mom[c, 1:4] == sp[f, :3].astype(np.float32))
    # root = global moments
    assert abs(mom[0, 0] - m.astype(np.float64).sum()) < 1e-6 * m.sum()


def test_parallel_axis_identity_child_to_parent():
    pos, m = _inputs("plummer", 4096)
    t = oracle.Tree(pos, m)
    cells, mom = t.cells(), t.moments().astype(np.float64)
    for c in np.flatnonzero(cells[:, 3] >= 0)[:200]:
        ch = np.arange(cells[c, 3], cells[c, 3] + cells[c, 4])
        M = mom[ch, 0].sum()
        com = (mom[ch, 0:1] * mom[ch, 1:4]).sum(0) / M
        d = mom[ch, 1:4] - com
        qxx = (mom[ch, 4] + mom[ch, 0] * d[:, 0] ** 2).sum()
        qxy = (mom[ch, 7] + mom[ch, 0] * d[:, 0] * d[:, 1]).sum()
        tr = mom[c, 4] + mom[c, 5] + mom[c, 6]
        assert abs(mom[c, 4] - qxx) <= 1e-6 * tr and abs(mom[c, 7] - qxy) <= 1e-6 * tr


def test_groups_are_runs_of_64_with_tight_boxes():
    pos, m = _inputs("plummer", 1000)  # ragged last group: 1000 = 15*64 + 40
    t = oracle.Tree(pos, m)
    assert t.n_groups == 16
    sp = t.sorted_particles()
    gmin, gmax = t.groups()
    for g in range(16):
        x = sp[64 * g: min(64 * g + 64, 1000), :3]
        assert np.array_equal(gmin[g], x.min(0)) and np.array_equal(gmax[g], x.max(0))
