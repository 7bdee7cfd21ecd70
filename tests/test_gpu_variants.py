"""The packed FP32x2 evaluators (FADD2 / FMUL2 / FFMA2, two targets per lane) against the scalar evaluators: the same
IEEE operations in the same order, so a build with -DBH_PACKED=0 must return the same BYTES (DESIGN.md section 5,
"Packed FP32x2 evaluators").  Builds the scalar variant with nvcc on the GPU box and runs both libraries in their own
processes (BHTREE_LIB selects the library the binding loads)."""
import os
import shutil
import subprocess
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_RUN = r"""
import sys, numpy as np, torch
from nbody_inputs import plummer, milky_way
from paper_1412_0659_b200 import Tree
out = sys.argv[1]
res = {}
for name, gen, n, eps in (("plummer", plummer, 40000, 0.01), ("mw", milky_way, 50011, 0.01)):
    pos, _, mass = gen(n, 11, with_vel=False)
    t = Tree(device=0, leaf_size=16, group_size=64)
    acc = torch.empty((n, 3), device="cuda"); pot = torch.empty(n, device="cuda")
    t.build(pos.cuda(), mass.cuda())
    t.force(0.4, eps, acc, pot)
    torch.cuda.synchronize()
    res[name + "_acc"] = acc.cpu().numpy(); res[name + "_pot"] = pot.cpu().numpy()
    res[name + "_counts"] = t.debug("counts")
np.savez(out, **res)
"""


def _run(lib, out):
    env = dict(os.environ)
    env["PYTHONPATH"] = ROOT + os.pathsep + env.get("PYTHONPATH", "")
    if lib:
        env["BHTREE_LIB"] = str(lib)
    else:
        env.pop("BHTREE_LIB", None)
    r = subprocess.run([sys.executable, "-c", _RUN, str(out)], env=env, cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    return np.load(out)


def test_packed_and_scalar_evaluators_return_the_same_bytes(tmp_path):
    from paper_1412_0659_b200 import build
    if shutil.which(build._nvcc()) is None and not os.path.exists(build._nvcc()):
        pytest.skip("no nvcc on this box")
    scalar = build.build_variant(tmp_path / "libbhtree_scalar.so", ["-DBH_PACKED=0"])
    a = _run(None, tmp_path / "packed.npz")
    b = _run(scalar, tmp_path / "scalar.npz")
    for k in a.files:
        assert a[k].tobytes() == b[k].tobytes(), k
    assert np.isfinite(a["plummer_acc"]).all() and np.abs(a["mw_pot"]).min() > 0
