"""Pins for the fp64 oracle (oracle/): things the paper and the mathematics fix.

Each test is chosen so that a plausible mistake in oracle/flashvan_oracle.c (dropped term,
wrong sign/index, transposed operand, look-ahead leak) fails at least one of them.
Pin numbering follows SURVEY.md 8(c-3) / DESIGN.md.
"""
import dataclasses
import itertools
import math
import os

import numpy as np
import pytest
import torch
import torch.nn.functional as F

from oracle import oracle as O
from paper_2606_22984_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def all_configs(n):
    return np.array(list(itertools.product([-1, 1], repeat=n)), dtype=np.int8)


def tiny(n=8, d=16, heads=2, layers=2, window=0, **kw):
    return dataclasses.replace(W.CONFIGS["cfg1"], name="tiny", L=n, n_sites=n, d_model=d,
                               n_heads=heads, n_layers=layers, window=window, batch=64, **kw)


# ---------------------------------------------------------------- P1: parameter inventory
def test_p1_param_counts_match_paper():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "param_counts.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 14
    for count, vocab, n_seq, d_token, d_model, n_layers in (map(int, r) for r in rows):
        assert O.param_count(vocab, n_seq, d_token, d_model, n_layers) == count
        # variants the paper's numbers exclude: an output projection, a 3-token vocabulary
        assert O.param_count(vocab, n_seq, d_token, d_model, n_layers, has_wo=1) != count
        assert O.param_count(vocab + 1, n_seq, d_token, d_model, n_layers) != count
        if vocab == 2:      # the blob the oracle actually carves has exactly that many entries
            w = dataclasses.replace(W.CONFIGS["cfg1"], n_sites=n_seq, L=n_seq, d_model=d_model,
                                    n_layers=n_layers, d_token=d_token)
            assert O.n_weights(w) + n_seq * (d_model - d_token) == count
            assert W.n_weights(w) == O.n_weights(w)


# --------------------------------------------- library-op restatement (torch CPU, fp64)
def torch_forward(w, weights, posemb, rowptr, col, spins):
    """Independent restatement of Alg. 1 with torch library ops and a DENSE additive mask."""
    v = {k: torch.from_numpy(np.array(a, dtype=np.float64)) for k, a in W.weight_views(w, weights).items()}
    pos = torch.from_numpy(posemb.astype(np.float64))
    s = torch.from_numpy(spins.astype(np.int64))
    B, N = s.shape
    d, nh = w.d_model, w.n_heads
    dh = d // nh
    tok = torch.cat([torch.zeros(B, 1, dtype=torch.int64), (s[:, :-1] + 1) // 2], dim=1)
    x = torch.cat([v["tok_emb"][tok], pos.unsqueeze(0).expand(B, N, -1)], dim=-1)
    allow = torch.zeros(N, N, dtype=torch.bool)
    for t in range(N):
        allow[t, col[rowptr[t]:rowptr[t + 1]].astype(np.int64)] = True
    bias = torch.zeros(N, N, dtype=torch.float64).masked_fill(~allow, float("-inf"))
    for l in range(w.n_layers):
        p = f"l{l}."
        a = F.layer_norm(x, (d,), v[p + "ln1_g"], v[p + "ln1_b"], w.ln_eps)
        q = F.linear(a, v[p + "wq"], v[p + "bq"]).view(B, N, nh, dh).transpose(1, 2)
        k = F.linear(a, v[p + "wk"], v[p + "bk"]).view(B, N, nh, dh).transpose(1, 2)
        vv = F.linear(a, v[p + "wv"], v[p + "bv"]).view(B, N, nh, dh).transpose(1, 2)
        att = torch.softmax(q @ k.transpose(-1, -2) / math.sqrt(dh) + bias, dim=-1)
        u = (att @ vv).transpose(1, 2).reshape(B, N, d)
        if w.has_wo:
            u = F.linear(u, v[p + "wo"], v[p + "bo"])
        x = x + u
        a2 = F.layer_norm(x, (d,), v[p + "ln2_g"], v[p + "ln2_b"], w.ln_eps)
        if w.ln2_style == 1:
            x = a2
        x = x + F.linear(F.gelu(F.linear(a2, v[p + "w1"], v[p + "b1"])), v[p + "w2"], v[p + "b2"])
    z = F.linear(x, v["head_w"], v["head_b"])
    p_up = torch.sigmoid(z[..., 1] - z[..., 0])          # P10: softmax(z)[1] == sigmoid(z1 - z0)
    lp = torch.log_softmax(z, dim=-1)
    logq = torch.where(s > 0, lp[..., 1], lp[..., 0]).sum(-1)
    return logq.numpy(), p_up.numpy()


@pytest.mark.parametrize("variant", [dict(), dict(has_wo=1), dict(ln2_style=1)])
@pytest.mark.parametrize("name", ["cfg1", "ea2d", "ea3d"])
def test_p6_p10_library_restatement(name, variant):
    if name == "cfg1":
        w = dataclasses.replace(W.CONFIGS["cfg1"], **variant)
    elif name == "ea2d":
        w = dataclasses.replace(W.CONFIGS["cfg2"], L=6, n_sites=36, window=4, d_model=32, n_heads=2,
                                n_layers=2, **variant)
    else:
        w = dataclasses.replace(W.CONFIGS["cfg4"], L=3, n_sites=27, window=5, d_model=48, n_heads=3,
                                n_layers=2, **variant)
    wt = W.make_weights(w, std=0.3)                      # large weights: sharp, non-trivial softmaxes
    pe = W.make_posemb(w, std=0.5)
    rp, col = W.make_mask_csr(w)
    spins = W.make_spins(w, 5)
    lq, cp = O.log_prob(w, wt, pe, rp, col, spins)
    lq_t, cp_t = torch_forward(w, wt, pe, rp, col, spins)
    assert np.abs(cp - cp_t).max() < 1e-12
    assert np.abs(lq - lq_t).max() < 1e-10
    assert cp.std() > 0.05                               # the case is not degenerate


# ------------------------------------------------------------ P2/P4: brute force at N<=16
@pytest.fixture(scope="module")
def cfg1_enum():
    w = W.CONFIGS["cfg1"]
    inp = W.make_all(w)
    S = all_configs(w.n_sites)
    lq, _ = O.log_prob(w, inp["weights"], inp["posemb"], inp["mask_rowptr"], inp["mask_col"], S)
    E = O.energy_dense(S, inp["J"])
    return w, inp, S, lq, E


def test_p2_normalisation_cfg1_full_enumeration(cfg1_enum):
    _, _, _, lq, _ = cfg1_enum
    assert abs(np.exp(lq).sum() - 1.0) < 1e-12


@pytest.mark.parametrize("window", [0, 2, 3])
@pytest.mark.parametrize("variant", [dict(), dict(has_wo=1), dict(ln2_style=1)])
def test_p2_normalisation_sparse_masks(window, variant):
    if window == 0:
        w = tiny(10, **variant)
    else:
        w = dataclasses.replace(W.CONFIGS["cfg2"], L=3, n_sites=9, window=window, d_model=16,
                                n_heads=2, n_layers=2, **variant)
    wt, pe = W.make_weights(w, std=0.4), W.make_posemb(w, std=0.4)
    rp, col = W.make_mask_csr(w)
    lq, _ = O.log_prob(w, wt, pe, rp, col, all_configs(w.n_sites))
    assert abs(np.exp(lq).sum() - 1.0) < 1e-12
    assert np.exp(lq).std() > 1e-4                       # far from the uniform distribution


def test_p4_exact_observables_and_kl(cfg1_enum):
    w, inp, S, lq, E = cfg1_enum
    beta = 1.0
    q = np.exp(lq)
    Fq = float((q * (E + lq / beta)).sum())              # Eq. 5
    lnZ = float(np.logaddexp.reduce(-beta * E))
    Fex = -lnZ / beta
    lnp = -beta * E - lnZ                                # Eq. 1
    kl = float((q * (lq - lnp)).sum())                   # Eq. 4, direct
    assert kl >= 0.0
    assert abs(kl - beta * (Fq - Fex)) < 1e-10
    # the 1024 seeded samples reproduce the exact mean of L = E + T log q within 5 sigma
    spins, lq_s, _ = O.sample(w, inp["weights"], inp["posemb"], inp["mask_rowptr"], inp["mask_col"],
                              inp["uniforms"])
    Ls = O.energy_dense(spins, inp["J"]) + lq_s / beta
    var = float((q * (E + lq / beta - Fq) ** 2).sum())
    assert abs(Ls.mean() - Fq) < 5 * math.sqrt(var / len(Ls))
    mean, std = O.free_energy(O.energy_dense(spins, inp["J"]), lq_s, beta)
    assert abs(mean - Ls.mean()) < 1e-12 and abs(std - Ls.std()) < 1e-12


@pytest.mark.parametrize("beta", [0.5, 1.5])
def test_p4_free_energy_at_beta_not_one(cfg1_enum, beta):
    """`oracle.free_energy` at the two temperatures cfg3 is evaluated at.  At beta = 1, E + log q / beta and
    E + beta log q coincide, so only beta != 1 can tell Eq. 5 (F_q = sum_s q [E + ln q / beta])
    from a beta / T swap.  The exact value comes from the enumerated q and E, not from `free_energy`; the
    sample estimate must land within 5 sigma of it, and the swapped formula must not (so the pin can fail)."""
    w, inp, S, lq, E = cfg1_enum
    q = np.exp(lq)
    Fq = float((q * (E + lq / beta)).sum())
    lnZ = float(np.logaddexp.reduce(-beta * E))
    kl = float((q * (lq - (-beta * E - lnZ))).sum())     # Eq. 4 written out, no F_q in it
    assert kl >= 0.0 and abs(kl - beta * (Fq - (-lnZ / beta))) < 1e-10
    spins, lq_s, _ = O.sample(w, inp["weights"], inp["posemb"], inp["mask_rowptr"], inp["mask_col"],
                              inp["uniforms"])
    E_s = O.energy_dense(spins, inp["J"])
    mean, std = O.free_energy(E_s, lq_s, beta)
    sigma = math.sqrt(float((q * (E + lq / beta - Fq) ** 2).sum()))
    assert abs(mean - Fq) < 5 * sigma / math.sqrt(len(E_s))
    swapped = float((q * (E + lq * beta)).sum())         # what a beta <-> T mix-up would converge to
    assert abs(mean - swapped) > 20 * sigma / math.sqrt(len(E_s))
    assert abs(std - sigma) < 0.15 * sigma               # spread of L = E + T log q under q, from the enumeration


def test_free_energy_std_is_the_population_std():
    """Two samples with L = 0 and L = 2 at T = 2: mean 1, population std 1 (the ddof = 1 estimate would be
    sqrt 2).  The GPU kernel and shard.merge_free_energy are held to the same convention."""
    mean, std = O.free_energy(np.array([0.0, 4.0]), np.array([0.0, -1.0]), 0.5)
    assert mean == 1.0 and std == 1.0


# ----------------------------------------------------------------------- P3: chain rule
@pytest.mark.parametrize("name", ["cfg1", "ea2d"])
def test_p3_chain_rule_sample_equals_log_prob(name):
    w = W.CONFIGS["cfg1"] if name == "cfg1" else dataclasses.replace(
        W.CONFIGS["cfg2"], L=8, n_sites=64, window=4, d_model=32, n_heads=2, n_layers=3)
    wt, pe = W.make_weights(w, std=0.2), W.make_posemb(w, std=0.3)
    rp, col = W.make_mask_csr(w)
    u = W.make_uniforms(w, 48)
    spins, lq_s, cp_s = O.sample(w, wt, pe, rp, col, u)
    lq, cp = O.log_prob(w, wt, pe, rp, col, spins)
    assert np.abs(lq - lq_s).max() < 1e-12
    assert np.abs(cp - cp_s).max() < 1e-13
    assert np.array_equal(spins, np.where(u < cp, 1, -1))        # draw rule, reading A10
    picked = np.where(spins > 0, cp, 1 - cp)
    assert np.abs(np.log(picked).sum(1) - lq).max() < 1e-11


# --------------------------------------------------------------------- P5: mask locality
def test_p5_self_only_mask_is_first_order_markov():
    w = tiny(9, layers=3)
    wt, pe = W.make_weights(w, std=0.4), W.make_posemb(w, std=0.4)
    rp = np.arange(w.n_sites + 1, dtype=np.int32)
    col = np.arange(w.n_sites, dtype=np.int32)               # A(t) = {t}
    S = all_configs(w.n_sites)
    lq, cp = O.log_prob(w, wt, pe, rp, col, S)
    assert abs(np.exp(lq).sum() - 1.0) < 1e-12
    for t in range(1, w.n_sites):                            # p_t depends on s_{t-1} only
        for prev in (-1, 1):
            vals = cp[S[:, t - 1] == prev, t]
            assert vals.max() - vals.min() == 0.0
    assert cp[:, 0].max() - cp[:, 0].min() == 0.0


def test_p5_receptive_field_closure():
    w = dataclasses.replace(W.CONFIGS["cfg2"], L=6, n_sites=36, window=2, d_model=32, n_heads=2, n_layers=2)
    wt, pe = W.make_weights(w, std=0.3), W.make_posemb(w, std=0.3)
    rp, col = W.make_mask_csr(w)
    N = w.n_sites
    reach = [set([t]) for t in range(N)]                     # positions reachable in n_l hops
    for _ in range(w.n_layers):
        reach = [set().union(*[set(col[rp[p]:rp[p + 1]].tolist()) for p in r]) | r for r in reach]
    base = W.make_spins(w, 1)
    _, cp0 = O.log_prob(w, wt, pe, rp, col, base)
    n_out = n_in = 0
    for j in range(N - 1):
        flipped = base.copy()
        flipped[0, j] *= -1                                  # spin j enters at position j+1
        _, cp1 = O.log_prob(w, wt, pe, rp, col, flipped)
        for t in range(N):
            if (j + 1) not in reach[t]:
                assert cp1[0, t] == cp0[0, t]
                n_out += 1
            elif cp1[0, t] != cp0[0, t]:
                n_in += 1
    assert n_out > 100 and n_in > 100
    assert np.array_equal(np.triu(np.ones((N, N)), 1) * 0, np.zeros((N, N)))  # (shape sanity)


# --------------------------------------------------------------------------- P7: energy
def test_p7_energy_closed_forms():
    rng = np.random.default_rng(5)
    for w in (dataclasses.replace(W.CONFIGS["cfg2"], L=5, n_sites=25),
              dataclasses.replace(W.CONFIGS["cfg4"], L=4, n_sites=64),
              dataclasses.replace(W.CONFIGS["cfg4"], L=3, n_sites=27, coupling="pm1")):
        rp, col, val = W.make_couplings_ea(w)
        assert rp[-1] == w.dim * w.n_sites
        S = (2 * rng.integers(0, 2, size=(33, w.n_sites)) - 1).astype(np.int8)
        E = O.energy_csr(S, rp, col, val)
        Jd = W.csr_to_dense_sym(w.n_sites, rp, col, val)
        Sf = S.astype(np.float64)
        assert np.abs(E + 0.5 * np.einsum("bi,ij,bj->b", Sf, Jd, Sf)).max() < 1e-10   # -1/2 s^T J s
        assert np.abs(E - O.energy_dense(S, Jd.astype(np.float32))).max() < 1e-10     # double loop
        assert np.array_equal(E, O.energy_csr(-S, rp, col, val))                       # E(s) = E(-s)
        ferro = O.energy_csr(np.ones((1, w.n_sites), np.int8), rp, col, np.ones_like(val))
        assert ferro[0] == -w.dim * w.n_sites                                          # -D N
        if w.coupling == "pm1":
            assert np.all(E == np.round(E)) and np.all((E.astype(np.int64) - rp[-1]) % 2 == 0)
    n, c = 12, 0.37
    J = np.full((n, n), c, np.float32)
    np.fill_diagonal(J, 0)
    S = all_configs(n)
    M = S.sum(1).astype(np.float64)
    assert np.abs(O.energy_dense(S, J) + np.float32(c).astype(np.float64) * (M * M - n) / 2).max() < 1e-9
    one = np.zeros((4, 4), np.float32)
    one[1, 2] = 2.0                                           # only the i<j triangle is read
    assert O.energy_dense(np.array([[1, 1, -1, 1]], np.int8), one)[0] == 2.0


# --------------------------------------------------------------- P8: degenerate weights
def test_p8_zero_weights_give_half():
    w = tiny(7)
    wt = np.zeros(W.n_weights(w), np.float32)
    pe = W.make_posemb(w)
    rp, col = W.make_mask_csr(w)
    S = W.make_spins(w, 6)
    lq, cp = O.log_prob(w, wt, pe, rp, col, S)
    assert np.all(cp == 0.5) and np.abs(lq + w.n_sites * math.log(2)).max() < 1e-14
    u = W.make_uniforms(w, 6)
    spins, lq_s, _ = O.sample(w, wt, pe, rp, col, u)
    assert np.array_equal(spins, np.where(u < 0.5, 1, -1))
    assert np.abs(lq_s + w.n_sites * math.log(2)).max() < 1e-14


def test_head_bias_only_closed_form():
    """With every matrix zero, h is the embedding and z = head_b: p = sigmoid(b1 - b0)."""
    w = tiny(5)
    wt = np.zeros(W.n_weights(w), np.float32)
    v = W.weight_views(w, wt)
    v["head_b"][:] = (0.3, -0.9)
    rp, col = W.make_mask_csr(w)
    _, cp = O.log_prob(w, wt, W.make_posemb(w), rp, col, W.make_spins(w, 3))
    b = v["head_b"].astype(np.float64)
    assert np.abs(cp - 1.0 / (1.0 + math.exp(b[0] - b[1]))).max() < 1e-15


# ------------------------------------------------------------------- P9: SK convention
def test_p9_sk_normalisation():
    beta, T = 0.5, 2.0
    assert abs((-T * math.log(2) - beta / 4) - (-1.5112)) < 1e-4
    n = 12
    S = all_configs(n)
    w = dataclasses.replace(W.CONFIGS["cfg1"], L=n, n_sites=n)
    lnZ = []
    for seed in range(24):
        J = W.make_couplings_sk(w, seed=seed)
        assert np.array_equal(J, J.T) and np.all(np.diag(J) == 0)
        lnZ.append(np.logaddexp.reduce(-beta * O.energy_dense(S, J)))
    annealed = n * math.log(2) + beta ** 2 * (n - 1) / 4               # ln E[Z], var(J) = 1/N
    assert np.mean(lnZ) <= annealed + 1e-9                              # Jensen
    assert abs(np.mean(lnZ) - annealed) < 0.1                           # high-T: nearly tight
