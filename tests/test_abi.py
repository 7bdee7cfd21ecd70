"""CPU-only checks of the boundary: libbhtree.so builds, loads and exports every symbol that
include/tree.h declares (no compute calls without a GPU), and the host-side accounting helpers."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    txt = open(os.path.join(ROOT, "include", "tree.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(tree_[a-z0-9_]+)\s*\(", txt)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_1412_0659_b200 import build as b
    import paper_1412_0659_b200 as pkg
    b.build()
    lib = pkg.load_library()
    names = _declared()
    assert {"tree_create", "tree_build", "tree_force", "tree_leapfrog", "tree_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    assert set(pkg.exported_symbols()) == set(names)


def test_sass_is_sm100a_only():
    import subprocess
    import paper_1412_0659_b200 as pkg
    out = subprocess.run(["cuobjdump", "-lelf", str(pkg.library_path())], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_null_and_argument_errors_without_gpu():
    import ctypes as C
    import paper_1412_0659_b200 as pkg
    lib = pkg.load_library()
    assert lib.tree_create(None, 0, None, 16, 64) == -1
    h = C.c_void_p()
    assert lib.tree_create(C.byref(h), 0, None, 0, 64) == -1      # leaf size
    assert lib.tree_create(C.byref(h), 0, None, 16, 48) == -1     # group size
    assert lib.tree_build(None, None, None, 10) == -1
    assert lib.tree_force(None, 0.4, 0.01, None, None) == -1
    assert lib.tree_leapfrog(None, 0.1) == -1
    assert lib.tree_destroy(None) == -1
    assert lib.tree_last_error(None) == b""


def test_flop_convention_matches_paper_table2():
    # PAPER.md L190-192 + Table II "1 GPU" column: 13e6 x (1745*23 + 4529*65) / 2.45 s = 1.77 Tflops
    from paper_1412_0659_b200 import effective_flops
    vals = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "paper_table2_1gpu.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            vals[k] = float(v)
    per_particle = effective_flops(vals["pp_per_particle"], vals["pc_per_particle"])
    assert per_particle == 334520
    tflops = vals["n_particles"] * per_particle / vals["gravity_seconds"] / 1e12
    assert abs(tflops - vals["gpu_tflops"]) < 0.01


def test_no_product_import_of_oracle():
    # the product path must never route through oracle/ (or any CPU fallback)
    pat = re.compile(r"^\s*(import\s+oracle|from\s+oracle|#include\s*[<\"].*oracle)", re.M)
    for top in ("paper_1412_0659_b200", "nbody_inputs"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, top)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".h")):
                    assert not pat.search(open(os.path.join(dirpath, f)).read()), f
    # and the oracle never imports the CUDA package
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            assert "paper_1412_0659_b200" not in open(os.path.join(ROOT, "oracle", f)).read(), f


def test_bhtree_lib_names_the_library_and_a_missing_one_raises(tmp_path):
    # BHTREE_LIB selects another build of the library (tests/test_gpu_variants.py); there is still no fallback
    import subprocess, sys, os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    code = ("from paper_1412_0659_b200 import binding\n"
            "print(binding.library_path())\n"
            "try:\n    binding.load_library()\nexcept RuntimeError as e:\n    print('raised', 'no CPU fallback' in str(e))\n")
    env = dict(os.environ, BHTREE_LIB=str(tmp_path / "nothing.so"), PYTHONPATH=root)
    r = subprocess.run([sys.executable, "-c", code], env=env, cwd=root, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-1000:]
    out = r.stdout.strip().splitlines()
    assert out[0].endswith("nothing.so") and out[1] == "raised True"
