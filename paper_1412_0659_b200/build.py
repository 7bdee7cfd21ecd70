"""Build libbhtree.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1412_0659_b200.build [--force]

nvcc cross-compiles without a GPU.  bh_build.cu is compiled with -fmad=false so that every FP
operation feeding an integer decision or a stored moment is one IEEE operation (S9, S13);
bh_force.cu keeps FMA contraction (explicit fmaf where the order is part of the contract).
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "libbhtree.so"
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]
UNITS = {
    "bh_build.cu": ["-fmad=false"],
    "bh_force.cu": [],
    "bh_measure.cu": [],
    "bh_api.cu": [],
    "bh_noalloc.cu": [],
}


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.sep not in c or os.path.exists(c)):
            return c
    return "nvcc"


def needs_build() -> bool:
    if not LIB.exists():
        return True
    m = LIB.stat().st_mtime
    srcs = list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")) + [HERE.parent / "include" / "tree.h"]
    return any(s.stat().st_mtime > m for s in srcs)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    objdir = HERE / "build"
    objdir.mkdir(exist_ok=True)
    objs = []
    for src, extra in UNITS.items():
        obj = objdir / (src + ".o")
        cmd = [_nvcc(), *ARCH, *COMMON, *extra, "-c", str(CSRC / src), "-o", str(obj)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        (objdir / (src + ".ptxas.txt")).write_text(r.stderr)
        if verbose or r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError(f"nvcc failed on {src}")
        objs.append(str(obj))
    tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
    r = subprocess.run([_nvcc(), *ARCH, "-shared", "-o", str(tmp), *objs], capture_output=True, text=True)
    if r.returncode:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("link failed")
    os.replace(tmp, LIB)
    return LIB


def build_variant(out: Path, defines: list[str]) -> Path:
    """Build the same library with extra -D switches (e.g. ``["-DBH_PACKED=0"]``: scalar evaluators) into ``out``;
    load it with the environment variable BHTREE_LIB.  Objects go next to ``out``."""
    out = Path(out)
    objs = []
    for src, extra in UNITS.items():
        obj = out.parent / (out.stem + "." + src + ".o")
        cmd = [_nvcc(), *ARCH, *COMMON, *extra, *defines, "-c", str(CSRC / src), "-o", str(obj)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError(f"nvcc failed on {src}")
        objs.append(str(obj))
    r = subprocess.run([_nvcc(), *ARCH, "-shared", "-o", str(out), *objs], capture_output=True, text=True)
    if r.returncode:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("link failed")
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
