"""Pins of the patch-token oracle (oracle.tok_sample / tok_log_prob / tokens_to_spins, SI I.D:
one token per 2^D-spin patch, vocabulary 2^(2^D), sequence (L/2)^D) -- no GPU needed.  The oracle is held to
what the paper and the mathematics fix: the parameter counts printed for the patched models, normalisation by
brute force over all 16^4 token sequences, the chain rule over two loop structures, the inverse-CDF draw rule
re-derived in numpy from the returned distributions, the reduction to the (separately pinned) one-spin-per-token
oracle at V = 2, the closed form at zero weights, and the bit <-> lattice-site unpacking."""
import dataclasses
import itertools
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_22984_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "param_counts.txt")


def small_patched(**kw):
    base = dataclasses.replace(W.CONFIGS["cfg2"], L=4, n_sites=16, window=2, d_model=16, n_heads=2, n_layers=2, **kw)
    return W.patched(base)


def test_patched_parameter_counts_printed_in_the_paper():
    """Table 7 "w/ patch" and l.670: the blob the oracle carves for V = 16 plus the position
    table has exactly the printed number of parameters."""
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    checked = 0
    for count, vocab, n_seq, d_token, d_model, n_layers in (map(int, r) for r in rows):
        if vocab == 2 or d_model % 16:
            continue
        Lt = int(round(math.sqrt(n_seq)))
        w = dataclasses.replace(W.CONFIGS["cfg2"], L=Lt, n_sites=n_seq, d_model=d_model, n_heads=1, n_layers=n_layers,
                                d_token=d_token, vocab=vocab, patch=2)
        assert O.n_weights(w) + n_seq * w.d_pos == count
        assert W.n_weights(w) == O.n_weights(w)
        checked += 1
    assert checked >= 6


def test_normalisation_by_enumeration_of_all_token_sequences():
    w = small_patched()
    wt, pe = W.make_weights(w, std=0.5), W.make_posemb(w, std=0.5)
    rp, col = W.make_mask_csr(w)
    seqs = np.array(list(itertools.product(range(w.vocab), repeat=w.n_sites)), dtype=np.int32)     # 16^4
    lq, _ = O.tok_log_prob(w, wt, pe, rp, col, seqs)
    q = np.exp(lq)
    assert abs(q.sum() - 1.0) < 1e-12
    assert q.std() > 1e-6 * q.mean()                       # not the uniform distribution


def test_chain_rule_and_inverse_cdf_draw():
    w = dataclasses.replace(small_patched(), L=3, n_sites=9)        # 6 x 6 spins, 9 tokens
    wt, pe = W.make_weights(w, std=0.12), W.make_posemb(w, std=0.3)
    rp, col = W.make_mask_csr(w)
    u = W.make_uniforms(w, 64, seed=5)
    tok, lq, pr = O.tok_sample(w, wt, pe, rp, col, u)
    lq2, pr2 = O.tok_log_prob(w, wt, pe, rp, col, tok)
    assert np.abs(lq - lq2).max() < 1e-12 and np.abs(pr - pr2).max() < 1e-12
    assert np.abs(pr.sum(-1) - 1.0).max() < 1e-12 and (pr > 0).all()
    # the draw rule, from the returned distributions: first k with u < p_0 + .. + p_k
    cdf = np.cumsum(pr, axis=-1)
    want = np.minimum((u.astype(np.float64)[..., None] >= cdf).sum(-1), w.vocab - 1)
    assert np.array_equal(tok, want)
    picked = np.take_along_axis(pr, tok[..., None], axis=-1)[..., 0]
    assert np.abs(np.log(picked).sum(1) - lq).max() < 1e-12
    assert len(np.unique(tok)) > 8                          # the draws spread over the vocabulary


def test_vocab_two_reduces_to_the_spin_oracle():
    """V = 2 is the one-spin-per-token model: same blob, and log q of a token sequence equals the (separately
    pinned) binary oracle's log q of the spins 2 token - 1."""
    w = dataclasses.replace(W.CONFIGS["cfg2"], L=4, n_sites=16, window=3, d_model=32, n_heads=2, n_layers=2)
    wt, pe = W.make_weights(w, std=0.3), W.make_posemb(w, std=0.3)
    rp, col = W.make_mask_csr(w)
    tok = W.make_tokens(w, 40)
    lq_t, pr = O.tok_log_prob(w, wt, pe, rp, col, tok)
    lq_s, cp = O.log_prob(w, wt, pe, rp, col, (2 * tok - 1).astype(np.int8))
    assert np.abs(lq_t - lq_s).max() < 1e-12
    assert np.abs(pr[..., 1] - cp).max() < 1e-13


def test_zero_weights_give_the_uniform_distribution():
    w = small_patched()
    wt = np.zeros(W.n_weights(w), np.float32)
    rp, col = W.make_mask_csr(w)
    lq, pr = O.tok_log_prob(w, wt, W.make_posemb(w), rp, col, W.make_tokens(w, 5))
    assert np.abs(lq + w.n_sites * math.log(w.vocab)).max() < 1e-12
    assert np.abs(pr - 1.0 / w.vocab).max() < 1e-15


@pytest.mark.parametrize("dim,L", [(2, 6), (3, 4)])
def test_token_bits_to_lattice_spins(dim, L):
    base = dataclasses.replace(W.CONFIGS["cfg2" if dim == 2 else "cfg4"], L=L, n_sites=L ** dim, window=2)
    w = W.patched(base)
    assert w.vocab == 2 ** (2 ** dim) and w.n_sites == (L // 2) ** dim
    si = W.patch_site_index(w)
    assert sorted(si.ravel().tolist()) == list(range(L ** dim))              # a partition of the lattice
    # every patch is a 2^dim block: the sites of one token differ from its first site by offsets in {0, 1}^dim
    strides = np.array([L ** (dim - 1 - a) for a in range(dim)])
    offs = sorted(int((np.array(o) * strides).sum()) for o in itertools.product(range(2), repeat=dim))
    assert all(sorted((si[n] - si[n, 0]).tolist()) == offs for n in range(w.n_sites))
    # one bit set -> exactly one up spin, at the listed site
    tok = np.zeros((1, w.n_sites), np.int32)
    tok[0, 3] = 1 << 2
    s = O.tokens_to_spins(tok, si)
    assert s.shape == (1, L ** dim) and (s == 1).sum() == 1 and s[0, si[3, 2]] == 1
    # all bits set everywhere -> ferromagnetic state: E = -D N on the periodic lattice with J = +1
    sl = W.spin_lattice(w)
    rp, col, val = W.make_couplings_ea(sl)
    s = O.tokens_to_spins(np.full((2, w.n_sites), w.vocab - 1, np.int32), si)
    E = O.energy_csr(s, rp, col, np.ones_like(val))
    assert (E == -dim * L ** dim).all()
