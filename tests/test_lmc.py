"""Local Monte Carlo sweeps (acceptance rule and sweep count not given in the paper:
parity with the authors' procedure is unpinned).  Pins of the oracle against the mathematics (no GPU)."""
import dataclasses
import itertools

import numpy as np

from oracle import lmc as OL
from oracle import oracle as O
from paper_2606_22984_b200 import workloads as W


def _setup(name="cfg2", L=6, coupling=None):
    w = dataclasses.replace(W.CONFIGS[name], L=L, n_sites=L ** W.CONFIGS[name].dim)
    if coupling:
        w = dataclasses.replace(w, coupling=coupling)
    brp, bcol, bval = W.make_couplings_ea(w)
    return w, (brp, bcol, bval), OL.full_adjacency(w.n_sites, brp, bcol, bval)


def test_energy_bookkeeping_against_the_energy_routine():
    """E(after) - E(before) recomputed by the independent bond-loop energy equals what the accepted flips say:
    replay the sweep, summing dE = 2 s_i h_i (in fp64 here) over the flips that the sweep accepted."""
    for coupling in ("pm1", "gauss"):
        w, bonds, (rp, col, val) = _setup(coupling=coupling)
        rng = np.random.default_rng(1)
        B, N, K = 6, w.n_sites, 3
        s0 = W.make_spins(w, B, seed=2)
        ev = rng.exponential(size=(B, K, N)).astype(np.float32)
        s1, acc = OL.sweeps(s0, rp, col, val, 0.8, ev)
        E0, E1 = O.energy_csr(s0, *bonds), O.energy_csr(s1, *bonds)
        # replay one sample site by site with the energy routine itself as the judge of every flip
        s = s0[:1].copy()
        for k in range(K):
            for i in range(N):
                t = s.copy()
                t[0, i] = -t[0, i]
                dE = O.energy_csr(t, *bonds)[0] - O.energy_csr(s, *bonds)[0]
                if np.float32(np.float32(0.8) * np.float32(dE)) < ev[0, k, i]:
                    s = t
        assert np.array_equal(s[0], s1[0])
        assert abs(O.energy_csr(s, *bonds)[0] - E1[0]) < 1e-9
        assert acc.min() > 0 and not np.array_equal(s0, s1) and np.isfinite(E0).all()


def test_beta_zero_flips_every_spin_and_zero_variates_only_descend():
    w, bonds, (rp, col, val) = _setup()
    B, N = 5, w.n_sites
    s0 = W.make_spins(w, B, seed=4)
    ev = np.full((B, 1, N), 0.5, np.float32)
    s1, acc = OL.sweeps(s0, rp, col, val, 0.0, ev)                 # beta = 0: 0 < e always
    assert np.array_equal(s1, -s0) and (acc == N).all()
    zero = np.zeros((B, 12, N), np.float32)                        # e = 0 (u = 1): only dE < 0 is accepted
    s2, _ = OL.sweeps(s0, rp, col, val, 1.0, zero)
    E0, E2 = O.energy_csr(s0, *bonds), O.energy_csr(s2, *bonds)
    assert (E2 <= E0).all() and (E2 < E0).any()
    s3, acc3 = OL.sweeps(s2, rp, col, val, 1.0, zero[:, :1])       # converged: a local minimum, nothing moves
    assert (acc3 == 0).all() and np.array_equal(s3, s2)
    for b in range(B):
        for i in range(N):
            h = sum(val[e] * s2[b, col[e]] for e in range(rp[i], rp[i + 1]))
            assert s2[b, i] * h >= 0


def test_one_sweep_transition_matrix_on_four_sites():
    """Exact Metropolis sweep kernel P = P_0 P_1 P_2 P_3 on a 4-site ring with generic couplings: the oracle's
    empirical transition frequencies match it, and the Boltzmann distribution is stationary under it."""
    N, beta = 4, 0.7
    rng = np.random.default_rng(8)
    J = np.zeros((N, N))
    for i in range(N):
        J[i, (i + 1) % N] = J[(i + 1) % N, i] = rng.normal()
    rp = np.arange(0, 2 * N + 1, 2).astype(np.int32)
    col = np.array([x for i in range(N) for x in sorted([(i - 1) % N, (i + 1) % N])], np.int32)
    val = np.array([J[i, j] for i in range(N) for j in sorted([(i - 1) % N, (i + 1) % N])], np.float32)
    states = np.array(list(itertools.product((-1, 1), repeat=N)), dtype=np.int8)
    index = {tuple(s): k for k, s in enumerate(states)}
    energy = np.array([-0.5 * s @ J @ s for s in states.astype(np.float64)])
    P = np.eye(len(states))
    for i in range(N):
        Pi = np.zeros_like(P)
        for k, s in enumerate(states):
            t = s.copy()
            t[i] = -t[i]
            a = min(1.0, np.exp(-beta * (energy[index[tuple(t)]] - energy[k])))
            Pi[k, index[tuple(t)]] += a
            Pi[k, k] += 1 - a
        P = P @ Pi
    pi = np.exp(-beta * energy)
    pi /= pi.sum()
    assert np.abs(pi @ P - pi).max() < 1e-12                       # stationarity of the analytic kernel
    R = 4000
    start = np.repeat(states, R, axis=0)
    ev = rng.exponential(size=(len(start), 1, N)).astype(np.float32)
    end, _ = OL.sweeps(start, rp, col, val, beta, ev)
    emp = np.zeros_like(P)
    for k in range(len(states)):
        idx = [index[tuple(s)] for s in end[k * R:(k + 1) * R]]
        emp[k] = np.bincount(idx, minlength=len(states)) / R
    sigma = np.sqrt(np.maximum(P * (1 - P), 1e-6) / R)
    assert (np.abs(emp - P) < 5 * sigma + 1e-3).all()
