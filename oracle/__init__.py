"""ORACLE — test infrastructure, not product code.

Thin numpy/ctypes face of ``oracle/bh_oracle.cpp`` (plain CPU Barnes-Hut + O(N^2) direct sum
written from PAPER.md; see that file's header for what it follows and what pins it).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "bh_oracle.cpp"
_LIB = _HERE / "libbh_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (no CUDA). -ffp-contract=off: FMA only where written."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["g++", "-O3", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
               "-fPIC", "-shared", str(_SRC), "-o", str(tmp)]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        L.orc_hilbert_key.restype = C.c_uint64
        L.orc_hilbert_key.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, C.c_int]
        L.orc_num_threads.restype = C.c_int
        L.orc_tree_create.restype = C.c_void_p
        L.orc_tree_create.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int, C.c_int, C.POINTER(C.c_int)]
        L.orc_tree_destroy.argtypes = [C.c_void_p]
        L.orc_tree_n_cells.restype = C.c_int64
        L.orc_tree_n_cells.argtypes = [C.c_void_p]
        L.orc_tree_n_groups.restype = C.c_int64
        L.orc_tree_n_groups.argtypes = [C.c_void_p]
        L.orc_direct.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_int64, C.c_double,
                                 C.c_void_p, C.c_void_p]
        L.orc_eval_pc.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]
        L.orc_tree_get_grid.argtypes = [C.c_void_p] * 4 + [C.POINTER(C.c_int)]
        L.orc_tree_get_keys.argtypes = [C.c_void_p] * 4
        L.orc_tree_get_cells.argtypes = [C.c_void_p] * 2
        L.orc_tree_get_moments.argtypes = [C.c_void_p] * 2
        L.orc_tree_set_moments.argtypes = [C.c_void_p] * 2
        L.orc_tree_get_groups.argtypes = [C.c_void_p] * 3
        L.orc_tree_get_sorted.argtypes = [C.c_void_p] * 2
        L.orc_tree_force.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_void_p, C.c_void_p, C.c_int64, C.c_int64]
        L.orc_tree_get_counts.argtypes = [C.c_void_p] * 3
        L.orc_tree_get_ropen2.argtypes = [C.c_void_p] * 2
        L.orc_tree_abs_sum.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_void_p, C.c_int64, C.c_void_p]
        L.orc_tree_set_mac.argtypes = [C.c_void_p, C.c_int]
        L.orc_tree_set_mac_relative.argtypes = [C.c_void_p, C.c_float, C.c_void_p]
        L.orc_tree_get_tight.argtypes = [C.c_void_p] * 2
        L.orc_tree_walk_lists.argtypes = [C.c_void_p, C.c_float, C.c_int64, C.c_void_p, C.POINTER(C.c_int64),
                                          C.c_void_p, C.POINTER(C.c_int64)]
        L.orc_leapfrog.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_float, C.c_int,
                                   C.c_float, C.c_float, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_int,
                                   C.c_void_p]
        _lib = L
    return _lib


def _f32(a, shape=None):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float32))
    if shape is not None:
        a = a.reshape(shape)
    return a


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def num_threads() -> int:
    return int(lib().orc_num_threads())


def hilbert_key(ix: int, iy: int, iz: int, bits: int = 21) -> int:
    """T3 Peano-Hilbert key of integer grid coordinates with ``bits`` bits per dimension."""
    return int(lib().orc_hilbert_key(int(ix), int(iy), int(iz), int(bits)))


def direct(pos, mass, eps: float, targets=None):
    """O-direct: exact softened sum over all j != i in FP64. Returns (acc [nt,3], pot [nt])."""
    pos = _f32(pos, (-1, 3))
    mass = _f32(mass, (-1,))
    n = pos.shape[0]
    tg = None if targets is None else np.ascontiguousarray(np.asarray(targets, dtype=np.int64))
    nt = n if tg is None else tg.shape[0]
    acc = np.zeros((nt, 3), dtype=np.float64)
    pot = np.zeros(nt, dtype=np.float64)
    # eps is the FP32 value the tree path receives (tree_force takes a float), promoted.
    rc = lib().orc_direct(_p(pos), _p(mass), n, _p(tg), nt, float(np.float32(eps)), _p(acc), _p(pot))
    if rc:
        raise ValueError(f"orc_direct failed: {rc}")
    return acc, pot


def eval_pc(target, com, M, Q, eps: float):
    """One particle-cell interaction, Eqs. (1),(2) softened (S1). Q = xx,yy,zz,xy,xz,yz."""
    t = np.ascontiguousarray(np.asarray(target, dtype=np.float64))
    c = _f32(com)
    q = _f32(Q)
    acc = np.zeros(3, dtype=np.float64)
    phi = C.c_double(0.0)
    lib().orc_eval_pc(_p(t), _p(c), float(M), _p(q), float(np.float32(eps)), _p(acc), C.byref(phi))
    return acc, phi.value


class Tree:
    """O-tree: T1-T8 at construction, T9-T11 in :meth:`force`."""

    def __init__(self, pos, mass, leaf_size: int = 16, group_size: int = 64):
        self.pos = _f32(pos, (-1, 3))
        self.mass = _f32(mass, (-1,))
        self.n = self.pos.shape[0]
        err = C.c_int(0)
        self._h = lib().orc_tree_create(_p(self.pos), _p(self.mass), self.n, leaf_size, group_size, C.byref(err))
        if not self._h:
            raise ValueError(f"oracle tree build failed: {err.value}")
        self.group_size = group_size
        self.leaf_size = leaf_size
        self.n_cells = int(lib().orc_tree_n_cells(self._h))
        self.n_groups = int(lib().orc_tree_n_groups(self._h))

    def __del__(self):
        h = getattr(self, "_h", None)
        if h and _lib is not None:
            try:
                _lib.orc_tree_destroy(h)
            except Exception:  # interpreter shutdown
                pass
            self._h = None

    def grid(self):
        lo = np.zeros(3, np.float32); hi = np.zeros(3, np.float32); org = np.zeros(3, np.float32)
        k = C.c_int(0)
        lib().orc_tree_get_grid(self._h, _p(lo), _p(hi), _p(org), C.byref(k))
        return lo, hi, org, k.value

    def keys(self):
        """(key in caller order, order[s] = original index at sorted slot s, sorted keys)."""
        key = np.zeros(self.n, np.uint64); order = np.zeros(self.n, np.uint32); sk = np.zeros(self.n, np.uint64)
        lib().orc_tree_get_keys(self._h, _p(key), _p(order), _p(sk))
        return key, order, sk

    def cells(self):
        """int32 [n_cells,5]: level, first, count, first_child (-1 = leaf), n_child. BFS order."""
        out = np.zeros((self.n_cells, 5), np.int32)
        lib().orc_tree_get_cells(self._h, _p(out))
        return out

    def moments(self):
        """float32 [n_cells,11]: M, cx, cy, cz, Qxx, Qyy, Qzz, Qxy, Qxz, Qyz, delta."""
        out = np.zeros((self.n_cells, 11), np.float32)
        lib().orc_tree_get_moments(self._h, _p(out))
        return out

    def set_moments(self, m):
        m = _f32(m, (self.n_cells, 11))
        lib().orc_tree_set_moments(self._h, _p(m))

    def groups(self):
        gmin = np.zeros((self.n_groups, 3), np.float32); gmax = np.zeros((self.n_groups, 3), np.float32)
        lib().orc_tree_get_groups(self._h, _p(gmin), _p(gmax))
        return gmin, gmax

    def sorted_particles(self):
        out = np.zeros((self.n, 4), np.float32)
        lib().orc_tree_get_sorted(self._h, _p(out))
        return out

    def force(self, theta: float, eps: float, g0: int = 0, stride: int = 1, out=None):
        """T9-T11. Returns acc [N,3] f64, pot [N] f64 (original order), n_pp, n_pc per group.
        ``out`` = (acc, pot) arrays to write into (entries of groups that are not walked are left as they are)."""
        if out is not None:
            acc, pot = out
            assert acc.shape == (self.n, 3) and pot.shape == (self.n,) and acc.dtype == np.float64 and pot.dtype == np.float64
        else:
            acc = np.zeros((self.n, 3), np.float64)
            pot = np.zeros(self.n, np.float64)
        rc = lib().orc_tree_force(self._h, float(theta), float(eps), _p(acc), _p(pot), int(g0), int(stride))
        if rc:
            raise ValueError(f"orc_tree_force failed: {rc}")
        npp = np.zeros(self.n_groups, np.uint32); npc = np.zeros(self.n_groups, np.uint32)
        lib().orc_tree_get_counts(self._h, _p(npp), _p(npc))
        return acc, pot, npp, npc

    def abs_sum(self, theta: float, eps: float, particles):
        """A_i = sum over particle i's interaction list of the magnitudes |a_ij| of its terms (diagnostic: A_i / |a_i| is
        the cancellation factor of the force sum).  ``particles``: caller indices.  Returns float64 [len(particles)]."""
        idx = np.asarray(particles, dtype=np.int64)
        inv = np.empty(self.n, np.int64)
        inv[self.keys()[1].astype(np.int64)] = np.arange(self.n, dtype=np.int64)
        slots = np.ascontiguousarray(inv[idx])
        out = np.zeros(len(slots), np.float64)
        if lib().orc_tree_abs_sum(self._h, float(theta), float(eps), _p(slots), len(slots), _p(out)):
            raise ValueError("orc_tree_abs_sum failed")
        return out

    def set_mac(self, kind: int):
        """Acceptance criterion of later force / walk_lists calls: 0 = canonical (S5), 1 = "bmax" (option, NEXT-2)."""
        if lib().orc_tree_set_mac(self._h, int(kind)):
            raise ValueError("unknown criterion")

    def set_mac_relative(self, alpha: float, amag):
        """Option "relative" (NEXT-2): group g accepts cell c iff the canonical criterion at the force call's theta does
        (the floor) and D^5 alpha a_g > M l^3, a_g = min of ``amag`` (float32 [N], caller order: |a| of every particle,
        an input) over the group's particles.  set_mac(0) returns to the canonical criterion."""
        amag = _f32(amag, (self.n,))
        if lib().orc_tree_set_mac_relative(self._h, float(alpha), _p(amag)):
            raise ValueError("bad alpha or amag")

    def tight(self):
        """float32 [n_cells,7]: tight bounding box lo, hi of each cell's particles and its bounding radius b."""
        out = np.zeros((self.n_cells, 7), np.float32)
        lib().orc_tree_get_tight(self._h, _p(out))
        return out

    def ropen2(self):
        out = np.zeros(self.n_cells, np.float32)
        lib().orc_tree_get_ropen2(self._h, _p(out))
        return out

    def walk_lists(self, theta: float, g: int):
        """(accepted cell ids, opened leaf ids) of group g for this theta (T10)."""
        a = np.zeros(self.n_cells, np.int32); o = np.zeros(self.n_cells, np.int32)
        na = C.c_int64(0); no = C.c_int64(0)
        rc = lib().orc_tree_walk_lists(self._h, float(theta), int(g), _p(a), C.byref(na), _p(o), C.byref(no))
        if rc:
            raise ValueError("bad group")
        return a[: na.value].copy(), o[: no.value].copy()


def leapfrog(pos, vel, mass, dt: float, nsteps: int, theta: float, eps: float,
             leaf_size: int = 16, group_size: int = 64, acc=None, pot=None):
    """T12: nsteps KDK steps with the tree force. Returns pos, vel, acc, pot (f32), energies [nsteps+1,2]."""
    pos = _f32(pos, (-1, 3)).copy(); vel = _f32(vel, (-1, 3)).copy(); mass = _f32(mass, (-1,))
    n = pos.shape[0]
    have = acc is not None and pot is not None
    a = _f32(acc, (-1, 3)).copy() if have else np.zeros((n, 3), np.float32)
    p = _f32(pot, (-1,)).copy() if have else np.zeros(n, np.float32)
    en = np.zeros((nsteps + 1, 2), np.float64)
    rc = lib().orc_leapfrog(_p(pos), _p(vel), _p(mass), n, float(dt), int(nsteps), float(theta), float(eps),
                            leaf_size, group_size, _p(a), _p(p), int(have), _p(en))
    if rc:
        raise ValueError(f"orc_leapfrog failed: {rc}")
    return pos, vel, a, p, en
