"""tree_energy_static (include/tree.h "an entry point that allocates nothing"): the energy sums from a static device
scratch array, checked against the existing path (tree_energy on a context) on two calls in a row.

Collected last on purpose (the file name): the suite runs with pytest -x, a failure here must not hide other tests.
"""
import ctypes as C

import pytest
import torch

import nbody_inputs as gen
from paper_1412_0659_b200 import ENERGY_STATIC_MAX_N, Tree, TreeError, load_library, tree_energy_static

# FP64 sums of the same FP32 terms in a different order (fixed-order partial sums here, atomic adds in arrival order in
# tree_energy): rounding only, ~1e-15 relative; the energy checks of tests/test_gpu_leapfrog_large.py resolve 1e-7.
REL = 1e-12


def test_size_beyond_the_static_scratch_is_rejected_with_a_clear_error():
    # sizes are checked before any CUDA call, so this needs no GPU
    lib = load_library()
    rc = lib.tree_energy_static(0, None, None, None, None, ENERGY_STATIC_MAX_N + 1, None)
    assert rc == -1
    msg = lib.tree_energy_static_error().decode()
    assert "TREE_ENERGY_STATIC_MAX_N" in msg and str(ENERGY_STATIC_MAX_N) in msg and "tree_energy" in msg
    assert lib.tree_energy_static(0, None, None, None, None, -1, None) == -1
    assert lib.tree_energy_static(64, None, None, None, None, 0, None) == -1


def _reference(n, seed, dev):
    """The existing path: state in a context, tree_energy; returns the caller-order arrays it was computed from."""
    pos, vel, mass = gen.plummer(n, seed, device=dev)
    t = Tree(device=0)
    t.build(pos, mass)
    t.set_velocity(vel)
    pot = torch.empty(n, dtype=torch.float32, device=dev)
    t.force(0.4, 0.01, None, pot)
    ke, pe = t.energy()
    t.close()
    return mass, vel, pot, ke, pe


@pytest.mark.gpu
def test_static_energy_matches_tree_energy_on_two_calls_in_a_row():
    dev = torch.device("cuda:0")
    stream = torch.cuda.current_stream().cuda_stream
    n1, n2 = 200_003, 50_001  # several blocks and a ragged tail; the second call uses fewer partial sums than the first
    mass1, vel1, pot1, ke1, pe1 = _reference(n1, 4101, dev)
    mass2, vel2, pot2, ke2, pe2 = _reference(n2, 4102, dev)
    tree_energy_static(0, stream, None, None, None, 0, None)  # set-up call
    out = torch.full((4, 2), float("nan"), dtype=torch.float64, device=dev)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # two calls in a row on the same inputs, then a smaller problem, then the first again: the scratch keeps the
    # previous call's partial sums and none of them may leak into the next result
    tree_energy_static(0, stream, mass1, vel1, pot1, n1, out[0])
    tree_energy_static(0, stream, mass1, vel1, pot1, n1, out[1])
    tree_energy_static(0, stream, mass2, vel2, pot2, n2, out[2])
    tree_energy_static(0, stream, mass1, vel1, pot1, n1, out[3])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0  # nothing was allocated on the device
    o = out.cpu().numpy()
    for k, (ke, pe) in enumerate([(ke1, pe1), (ke1, pe1), (ke2, pe2), (ke1, pe1)]):
        assert abs(o[k, 0] - ke) <= REL * abs(ke), (k, o[k, 0], ke)
        assert abs(o[k, 1] - pe) <= REL * abs(pe), (k, o[k, 1], pe)
    assert (o[0] == o[1]).all() and (o[0] == o[3]).all()  # fixed summation order: same bits on every call
    # virial sanity of the model (Plummer, G = M = a = 1): K = 3 pi / 64, W = -3 pi / 32 up to sampling and tree error
    assert abs(o[0, 0] / 0.147262 - 1) < 0.02 and abs(o[0, 1] / -0.294524 - 1) < 0.02


@pytest.mark.gpu
def test_static_energy_optional_inputs_and_argument_errors():
    dev = torch.device("cuda:0")
    stream = torch.cuda.current_stream().cuda_stream
    n = 10_000
    mass, vel, pot, ke, pe = _reference(n, 4103, dev)
    out = torch.full((2, 2), float("nan"), dtype=torch.float64, device=dev)
    tree_energy_static(0, stream, mass, None, pot, n, out[0])
    tree_energy_static(0, stream, mass, vel, None, n, out[1])
    torch.cuda.synchronize()
    o = out.cpu().numpy()
    assert o[0, 0] == 0.0 and abs(o[0, 1] - pe) <= REL * abs(pe)
    assert o[1, 1] == 0.0 and abs(o[1, 0] - ke) <= REL * abs(ke)
    with pytest.raises(TreeError, match="NULL"):
        tree_energy_static(0, stream, None, vel, pot, n, out[0])
    with pytest.raises(TreeError, match="TREE_ENERGY_STATIC_MAX_N"):
        tree_energy_static(0, stream, mass, vel, pot, ENERGY_STATIC_MAX_N + 1, out[0])
    assert load_library().tree_energy_static(0, C.c_void_p(stream), None, None, None, 0, None) == 0
    assert load_library().tree_energy_static_error() == b""
