"""GPU parity for the energy kernels and the F_q reduction (north_star tolerances)."""
import dataclasses

import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2606_22984_b200 import binding as fv
from paper_2606_22984_b200 import workloads as W

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("name,B", [("cfg2", 4096), ("cfg5", 257), ("cfg4", 1000)])
def test_energy_csr_full_size(name, B):
    w = W.CONFIGS[name]
    rp, col, val = W.make_couplings_ea(w)
    spins = W.make_spins(w, B, seed=3)
    E_o = O.energy_csr(spins, rp, col, val)
    integer = w.coupling == "pm1"
    E_g = fv.energy_csr(dev(spins), dev(rp), dev(col), dev(val), integer).cpu().numpy().astype(np.float64)
    if integer:
        assert np.array_equal(E_g, E_o)                                   # bit-exact integers
    else:
        scale = np.maximum(np.abs(E_o), np.sqrt((val.astype(np.float64) ** 2).sum()))
        assert (np.abs(E_g - E_o) <= 1e-4 * scale).all()
    # the float path on +-J couplings is exact as well (small integers in fp32)
    if integer:
        E_f = fv.energy_csr(dev(spins), dev(rp), dev(col), dev(val), False).cpu().numpy()
        assert np.array_equal(E_f.astype(np.float64), E_o)


def test_energy_csr_edge_cases():
    w = dataclasses.replace(W.CONFIGS["cfg2"], L=3, n_sites=9)
    rp, col, val = W.make_couplings_ea(w)
    for B in (1, 2, 33):
        s = W.make_spins(w, B, seed=B)
        E = fv.energy_csr(dev(s), dev(rp), dev(col), dev(val), True).cpu().numpy()
        assert np.array_equal(E.astype(np.float64), O.energy_csr(s, rp, col, val))
    ones = np.ones((2, 9), np.int8)
    E = fv.energy_csr(dev(ones), dev(rp), dev(col), dev(np.ones_like(val)), True).cpu().numpy()
    assert np.all(E == -18.0)                                              # ferromagnet: -D N


@pytest.mark.parametrize("N,B", [(16, 1024), (512, 300), (100, 77), (33, 5)])
def test_energy_dense(N, B):
    w = dataclasses.replace(W.CONFIGS["cfg3"], L=N, n_sites=N)
    J = W.make_couplings_sk(w)
    spins = W.make_spins(w, B, seed=4)
    E_o = O.energy_dense(spins, J)
    E_g = fv.energy_dense(dev(spins), dev(J)).cpu().numpy().astype(np.float64)
    scale = np.maximum(np.abs(E_o), np.sqrt((np.triu(J.astype(np.float64), 1) ** 2).sum()))
    assert (np.abs(E_g - E_o) <= 1e-4 * scale).all(), (np.abs(E_g - E_o) / scale).max()


def test_free_energy_reduction():
    rng = np.random.default_rng(9)
    E = rng.normal(-300, 20, size=5000).astype(np.float32)
    lq = rng.normal(-2800, 30, size=5000).astype(np.float32)
    for T in (1.0, 2.0, 1 / 1.5):
        mean, std = O.free_energy(E, lq, 1.0 / T)
        got = fv.free_energy(dev(E), dev(lq), T).cpu().numpy()
        assert abs(got[0] - mean) < 1e-9 * abs(mean) and abs(got[1] - std) < 1e-9 * std
