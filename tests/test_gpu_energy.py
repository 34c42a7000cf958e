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
        assert got[2] == len(E) and abs(got[3] - std * std * len(E)) < 1e-8 * got[3]
    with pytest.raises(fv.FlashVanError):                              # caller-supplied outputs are validated
        fv.free_energy(dev(E), dev(lq), 1.0, out=torch.empty(2, dtype=torch.float64, device="cuda"))
    with pytest.raises(fv.FlashVanError):
        fv.free_energy(dev(E), dev(lq), 1.0, out=torch.empty(4, dtype=torch.float64))


@pytest.mark.parametrize("B,N", [(1024, 4096), (257, 1000), (33, 17), (5, 1), (64, 16), (3, 4099)])
def test_overlap_matches_oracle_bit_exact(B, N):
    """Eq. 9: integer sums and the p(q) histogram, bit-exact (N a multiple of 16 or not: aligned vector path
    and byte tail; a row offset that breaks the alignment)."""
    rng = np.random.default_rng(B * 7919 + N)
    a = (rng.integers(0, 2, size=(B, N)) * 2 - 1).astype(np.int8)
    c = a.copy()
    flip = rng.random((B, N)) < rng.random((B, 1))            # per-sample flip rate: the whole range of q
    c[flip] *= -1
    dot_o, hist_o = O.overlap(a, c)
    dot_g, hist_g = fv.overlap(dev(a), dev(c))
    assert np.array_equal(dot_g.cpu().numpy().astype(np.int64), dot_o)
    assert np.array_equal(hist_g.cpu().numpy().astype(np.int64), hist_o)
    dot_g2, none = fv.overlap(dev(a), dev(a), want_hist=False)
    assert none is None and (dot_g2.cpu().numpy() == N).all()


def test_overlap_of_two_sampling_runs():
    """The paper's use: two independent sampling runs of one model (uniform seeds 1 and 2) -> q per replica pair."""
    w = dataclasses.replace(W.CONFIGS["cfg2"], L=8, n_sites=64)
    B = 96
    weights, posemb = W.make_weights(w), W.make_posemb(w)
    rp, col = W.make_mask_csr(w)
    model = fv.create_model(w, weights, rp, col, posemb, B)
    s1 = model.sample(dev(W.make_uniforms(w, B, 1)))[0].clone()
    s2 = model.sample(dev(W.make_uniforms(w, B, 2)))[0].clone()
    dot_g, hist_g = fv.overlap(s1, s2)
    dot_o, hist_o = O.overlap(s1.cpu().numpy(), s2.cpu().numpy())
    assert np.array_equal(dot_g.cpu().numpy().astype(np.int64), dot_o)
    assert np.array_equal(hist_g.cpu().numpy().astype(np.int64), hist_o) and int(hist_g.sum()) == B
    model.close()


@pytest.mark.parametrize("name,L,B,K,beta", [("cfg2", 8, 40, 3, 0.9), ("cfg4", 5, 33, 2, 1.7), ("cfg5", 64, 9, 1, 0.5),
                                              ("cfg2", 3, 5, 0, 1.0)])
def test_lmc_sweeps_match_oracle_bit_exact(name, L, B, K, beta):
    """Metropolis sweeps: every accept/reject is one fp32 product and one comparison on both sides, so the
    refined spins and the accepted-flip counts are bit-exact (+-J and Gaussian couplings, 2D and 3D, K = 0)."""
    from oracle import lmc as OL
    base = W.CONFIGS[name]
    w = dataclasses.replace(base, L=L, n_sites=L ** base.dim)
    N = w.n_sites
    brp, bcol, bval = W.make_couplings_ea(w)
    rp, col, val = OL.full_adjacency(N, brp, bcol, bval)
    spins = W.make_spins(w, B, seed=6)
    ev = np.random.default_rng(L * 100 + B).exponential(size=(B, K, N)).astype(np.float32)
    s_o, acc_o = OL.sweeps(spins, rp, col, val, beta, ev)
    s_g = dev(spins).clone()
    acc_g = fv.lmc_sweeps(s_g, dev(rp), dev(col), dev(val), beta, dev(ev))
    assert np.array_equal(s_g.cpu().numpy(), s_o)
    assert np.array_equal(acc_g.cpu().numpy().astype(np.int64), acc_o)
    if K:
        # the refined samples' energies, by the library's own energy kernel, against the reference's
        E_g = fv.energy_csr(s_g, dev(brp), dev(bcol), dev(bval), w.coupling == "pm1").cpu().numpy()
        E_o = O.energy_csr(s_o, brp, bcol, bval)
        assert np.allclose(E_g, E_o, rtol=1e-4, atol=1e-3)
