"""ctypes binding of include/tree.h — argument marshalling only.

torch is used for device memory and streams (``tensor.data_ptr()``, ``torch.cuda.current_stream``);
every step of the path runs inside libbhtree.so.
"""
from __future__ import annotations

import ctypes as C
import os
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
# BHTREE_LIB names another build of the same library (e.g. `build.build_variant`, used by the test that compares the
# packed and the scalar evaluators byte for byte); there is still no fallback: the named file must exist.
_LIBPATH = Path(os.environ["BHTREE_LIB"]).resolve() if os.environ.get("BHTREE_LIB") else _HERE / "libbhtree.so"
_lib = None

# Flop convention of PAPER.md L190-192: 23 per particle-particle, 65 per particle-cell interaction.
FLOP_PP = 23
FLOP_PC = 65
SHARD_MAX_WORLD = 16
SHARD_HANDLE_BYTES = 128

PHASES = ("keys", "sort", "permute", "build", "moments", "opening", "walk", "unpermute", "integrate", "sched", "total")

DBG = dict(keys=0, order=1, sorted_keys=2, cells=3, moments=4, group_boxes=5, counts=6, grid=7, ropen2=8,
           sorted_pos=9, level_offsets=10, task_trace=11, tight=12)
MAC_KINDS = dict(geometric=0, bmax=1)  # TREE_MAC_* of include/tree.h

_SIGS = {
    "tree_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_void_p, C.c_int, C.c_int]),
    "tree_build": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_longlong]),
    "tree_force": (C.c_int, [C.c_void_p, C.c_float, C.c_float, C.c_void_p, C.c_void_p]),
    "tree_leapfrog": (C.c_int, [C.c_void_p, C.c_float]),
    "tree_destroy": (C.c_int, [C.c_void_p]),
    "tree_set_velocity": (C.c_int, [C.c_void_p, C.c_void_p]),
    "tree_set_mac": (C.c_int, [C.c_void_p, C.c_int]),
    "tree_set_mac_relative": (C.c_int, [C.c_void_p, C.c_float, C.c_void_p]),
    "tree_get_state": (C.c_int, [C.c_void_p] * 5),
    "tree_build_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_longlong]),
    "tree_force_host": (C.c_int, [C.c_void_p, C.c_float, C.c_float, C.c_void_p, C.c_void_p]),
    "tree_direct": (C.c_int, [C.c_void_p, C.c_void_p, C.c_longlong, C.c_float, C.c_void_p, C.c_void_p]),
    "tree_energy": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "tree_get_debug": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.POINTER(C.c_longlong)]),
    "tree_get_stats": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(C.c_ulonglong), C.POINTER(C.c_ulonglong)]),
    "tree_reserve": (C.c_int, [C.c_void_p, C.c_longlong]),
    "tree_shard_config": (C.c_int, [C.c_void_p, C.c_int, C.c_int]),
    "tree_shard_export": (C.c_int, [C.c_void_p, C.c_void_p]),
    "tree_shard_attach": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "tree_shard_attach_local": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "tree_force_begin": (C.c_int, [C.c_void_p, C.c_float, C.c_float]),
    "tree_force_end": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "tree_leapfrog_begin": (C.c_int, [C.c_void_p, C.c_float]),
    "tree_leapfrog_mid": (C.c_int, [C.c_void_p]),
    "tree_leapfrog_end": (C.c_int, [C.c_void_p]),
    "tree_shard_range": (C.c_int, [C.c_void_p] + [C.POINTER(C.c_longlong)] * 4),
    "tree_fp32_peak": (C.c_int, [C.c_void_p, C.POINTER(C.c_double)]),
    "tree_measure_listeval": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "tree_energy_static": (C.c_int, [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_longlong, C.c_void_p]),
    "tree_energy_static_error": (C.c_char_p, []),
    "tree_launch_count": (C.c_longlong, [C.c_void_p]),
    "tree_last_error": (C.c_char_p, [C.c_void_p]),
}


class TreeError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libbhtree error {code}: {msg}")
        self.code = code


def library_path() -> Path:
    return _LIBPATH


def exported_symbols():
    return tuple(_SIGS)


def load_library():
    """Load libbhtree.so (built in-tree by ``python -m paper_1412_0659_b200.build``). No fallback."""
    global _lib
    if _lib is None:
        if not _LIBPATH.exists():
            raise RuntimeError(
                f"{_LIBPATH} is missing: build it with `python -m paper_1412_0659_b200.build` "
                "(there is no CPU fallback)")
        L = C.CDLL(str(_LIBPATH))
        for name, (res, args) in _SIGS.items():
            fn = getattr(L, name)  # AttributeError if a declared symbol is not exported
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _ptr(x):
    """Address of a torch tensor (device or host), a numpy array, an int address, or None."""
    if x is None:
        return None
    if isinstance(x, int):
        return C.c_void_p(x)
    if isinstance(x, np.ndarray):
        assert x.flags["C_CONTIGUOUS"]
        return C.c_void_p(x.ctypes.data)
    assert x.is_contiguous(), "tensor must be contiguous"
    return C.c_void_p(x.data_ptr())


def _check(handle, rc):
    if rc != 0:
        msg = load_library().tree_last_error(handle) if handle else b""
        raise TreeError(rc, (msg or b"").decode())


# ---- the five calls of north_star, same names as the C ABI -------------------------------
def tree_create(device: int = 0, stream=None, leaf_size: int = 16, group_size: int = 64):
    h = C.c_void_p()
    rc = load_library().tree_create(C.byref(h), int(device), _ptr(stream), int(leaf_size), int(group_size))
    if rc != 0:
        raise TreeError(rc, "tree_create failed")
    return h


def tree_build(h, pos, mass, n: int):
    _check(h, load_library().tree_build(h, _ptr(pos), _ptr(mass), int(n)))


def tree_force(h, theta: float, eps: float, acc=None, pot=None):
    _check(h, load_library().tree_force(h, float(theta), float(eps), _ptr(acc), _ptr(pot)))


def tree_leapfrog(h, dt: float):
    _check(h, load_library().tree_leapfrog(h, float(dt)))


def tree_destroy(h):
    load_library().tree_destroy(h)


ENERGY_STATIC_MAX_N = 134217728  # TREE_ENERGY_STATIC_MAX_N of include/tree.h


def tree_energy_static(device: int, stream, mass, vel, pot, n: int, out):
    """tree_energy_static: the energy sums without a context and without any allocation (static device scratch).
    mass [n], vel [n,3] or None, pot [n] or None: float32 device tensors; out: float64 device tensor [2]; n = 0: set-up."""
    rc = load_library().tree_energy_static(int(device), _ptr(stream), _ptr(mass), _ptr(vel), _ptr(pot), int(n), _ptr(out))
    if rc != 0:
        raise TreeError(rc, (load_library().tree_energy_static_error() or b"").decode())


def effective_flops(n_pp: int, n_pc: int) -> int:
    """flops = 23 * (number of p-p) + 65 * (number of p-c)."""
    return FLOP_PP * int(n_pp) + FLOP_PC * int(n_pc)


class Tree:
    """Convenience owner of one ``tree_ctx``; methods mirror the C ABI one to one."""

    def __init__(self, device: int = 0, stream=None, leaf_size: int = 16, group_size: int = 64):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1412_0659_b200 needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self.device = torch.device("cuda", device)
        if stream is None:
            stream = torch.cuda.current_stream(self.device).cuda_stream
        self.stream = int(stream)  # the cudaStream_t every call of this context enqueues on
        self.h = tree_create(device, self.stream, leaf_size, group_size)
        self.n = 0
        self.group_size = group_size
        self.leaf_size = leaf_size

    def close(self):
        if getattr(self, "h", None):
            tree_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- device-pointer calls
    def build(self, pos, mass):
        assert pos.is_cuda and mass.is_cuda and pos.dtype == self._torch.float32 and mass.dtype == self._torch.float32
        n = mass.numel()
        assert pos.numel() == 3 * n
        tree_build(self.h, pos, mass, n)
        self.n = n

    def force(self, theta: float, eps: float, acc=None, pot=None):
        tree_force(self.h, theta, eps, acc, pot)

    def leapfrog(self, dt: float):
        tree_leapfrog(self.h, dt)

    # -- sharded force pass (include/tree.h "sharded force pass"); ShardedTree in sharded.py drives these
    def reserve(self, n: int):
        _check(self.h, load_library().tree_reserve(self.h, int(n)))

    def shard_config(self, rank: int, world: int):
        _check(self.h, load_library().tree_shard_config(self.h, int(rank), int(world)))

    def shard_export(self) -> bytes:
        buf = C.create_string_buffer(SHARD_HANDLE_BYTES)
        _check(self.h, load_library().tree_shard_export(self.h, buf))
        return buf.raw

    def shard_attach(self, peer_rank: int, handle: bytes):
        assert len(handle) == SHARD_HANDLE_BYTES
        buf = C.create_string_buffer(handle, SHARD_HANDLE_BYTES)
        _check(self.h, load_library().tree_shard_attach(self.h, int(peer_rank), buf))

    def shard_attach_local(self, peer_rank: int, peer: "Tree"):
        _check(self.h, load_library().tree_shard_attach_local(self.h, int(peer_rank), peer.h))

    def force_begin(self, theta: float, eps: float):
        _check(self.h, load_library().tree_force_begin(self.h, float(theta), float(eps)))

    def force_end(self, acc=None, pot=None):
        _check(self.h, load_library().tree_force_end(self.h, _ptr(acc), _ptr(pot)))

    def leapfrog_begin(self, dt: float):
        _check(self.h, load_library().tree_leapfrog_begin(self.h, float(dt)))

    def leapfrog_mid(self):
        _check(self.h, load_library().tree_leapfrog_mid(self.h))

    def leapfrog_end(self):
        _check(self.h, load_library().tree_leapfrog_end(self.h))

    def shard_range(self):
        """(g_lo, g_hi, slot_lo, slot_hi) of the last pass on this context."""
        v = [C.c_longlong(0) for _ in range(4)]
        _check(self.h, load_library().tree_shard_range(self.h, *[C.byref(x) for x in v]))
        return tuple(int(x.value) for x in v)

    def set_mac(self, kind):
        """Acceptance criterion (tree_set_mac): 0 / "geometric" (default) or 1 / "bmax"; before build."""
        _check(self.h, load_library().tree_set_mac(self.h, int(MAC_KINDS.get(kind, kind))))

    def set_mac_relative(self, alpha: float, amag=None):
        """Error-targeted acceptance per group on top of the geometric criterion (tree_set_mac_relative); ``amag``: CUDA
        float32 [N] in caller order or None (the library's own last force pass)."""
        if amag is not None:
            assert amag.is_cuda and str(amag.dtype) == "torch.float32" and amag.is_contiguous() and (not self.n or amag.numel() == self.n)
        _check(self.h, load_library().tree_set_mac_relative(self.h, float(alpha), _ptr(amag)))

    def set_velocity(self, vel):
        assert vel.is_cuda and vel.numel() == 3 * self.n
        _check(self.h, load_library().tree_set_velocity(self.h, _ptr(vel)))

    def get_state(self, pos=None, vel=None, acc=None, pot=None):
        _check(self.h, load_library().tree_get_state(self.h, _ptr(pos), _ptr(vel), _ptr(acc), _ptr(pot)))

    # -- host-pointer calls (end-to-end path)
    def build_host(self, pos, mass):
        n = mass.numel() if hasattr(mass, "numel") else mass.size
        _check(self.h, load_library().tree_build_host(self.h, _ptr(pos), _ptr(mass), int(n)))
        self.n = int(n)

    def force_host(self, theta: float, eps: float, acc=None, pot=None):
        _check(self.h, load_library().tree_force_host(self.h, float(theta), float(eps), _ptr(acc), _ptr(pot)))

    def direct(self, idx, eps, acc, pot):
        """tree_direct: idx int64 device tensor [n]; acc float64 [n,3], pot float64 [n] device tensors."""
        _check(self.h, load_library().tree_direct(self.h, _ptr(idx), int(idx.numel()), float(eps), _ptr(acc), _ptr(pot)))

    def energy(self):
        ke, pe = C.c_double(0), C.c_double(0)
        _check(self.h, load_library().tree_energy(self.h, C.byref(ke), C.byref(pe)))
        return ke.value, pe.value

    def stats(self):
        ms = (C.c_double * len(PHASES))()
        pp, pc = C.c_ulonglong(0), C.c_ulonglong(0)
        _check(self.h, load_library().tree_get_stats(self.h, ms, C.byref(pp), C.byref(pc)))
        return dict(zip(PHASES, list(ms))), int(pp.value), int(pc.value)

    def fp32_peak(self) -> float:
        """Measured register-operand FFMA rate of this GPU in TFLOP/s (tree_fp32_peak)."""
        v = C.c_double(0)
        _check(self.h, load_library().tree_fp32_peak(self.h, C.byref(v)))
        return v.value

    def measure_listeval(self):
        """(walk-alone ms, evaluation-alone ms, max relative deviation from the fused pass): tree_measure_listeval."""
        ms = (C.c_double * 2)(); mr = C.c_double(0)
        _check(self.h, load_library().tree_measure_listeval(self.h, ms, C.byref(mr)))
        return ms[0], ms[1], mr.value

    def launch_count(self) -> int:
        return int(load_library().tree_launch_count(self.h))

    def debug(self, what: str) -> np.ndarray:
        code = DBG[what]
        cnt = C.c_longlong(0)
        _check(self.h, load_library().tree_get_debug(self.h, code, None, C.byref(cnt)))
        n = int(cnt.value)
        shape, dt = {
            "keys": ((n,), np.uint64), "order": ((n,), np.uint32), "sorted_keys": ((n,), np.uint64),
            "cells": ((n, 5), np.int32), "moments": ((n, 11), np.float32), "group_boxes": ((n, 6), np.float32),
            "counts": ((n, 2), np.uint32), "grid": ((n,), np.float32), "ropen2": ((n,), np.float32),
            "sorted_pos": ((n, 4), np.float32), "level_offsets": ((n,), np.int32),
            "task_trace": ((n, 4), np.uint32), "tight": ((n, 7), np.float32),
        }[what]
        out = np.zeros(shape, dt)
        _check(self.h, load_library().tree_get_debug(self.h, code, _ptr(out), C.byref(cnt)))
        return out
