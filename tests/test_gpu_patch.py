"""GPU parity of the patch-token path (SI I.D): fv_sample / fv_log_prob with vocab = 2^(2^D) and
fv_tokens_to_spins, against oracle.tok_log_prob / tokens_to_spins on the same seeded inputs.  Tolerances as for
the one-spin-per-token path: conditionals within 2e-3; the drawn token equals the oracle's inverse-CDF choice
(on the GPU's own token prefix) except where the uniform lies within 2e-3 of a boundary of the oracle's CDF --
those sites are counted and reported; the unpacked spins and their +-J energies are bit-exact."""
import dataclasses

import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2606_22984_b200 import binding as fv
from paper_2606_22984_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL_P = 2e-3


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


CASES = {
    "2d_L16_2x2": (dataclasses.replace(W.CONFIGS["cfg2"], window=3), 200),                                   # 64 tokens, V = 16, d = 64
    "2d_L8_2x2_d128": (dataclasses.replace(W.CONFIGS["cfg5"], L=8, n_sites=64, window=2, n_layers=3), 37),   # 16 tokens, d = 128
    "3d_L4_2x2x2": (dataclasses.replace(W.CONFIGS["cfg4"], L=4, n_sites=64, window=2, n_layers=2), 75),      # 8 tokens, V = 256
    "3d_L6_d32": (dataclasses.replace(W.CONFIGS["cfg4"], L=6, n_sites=216, window=3, n_layers=2, d_model=32, n_heads=2), 19),
}


@pytest.mark.parametrize("case", list(CASES))
def test_patch_tokens_against_oracle(case):
    base, B = CASES[case]
    w = W.patched(base)
    inp = W.make_all(w, batch=B)
    wt, pe, rp, col = inp["weights"], inp["posemb"], inp["mask_rowptr"], inp["mask_col"]
    model = fv.create_model(w, wt, rp, col, pe, B)
    V = w.vocab
    # ---- teacher-forced pass on random token sequences ----
    tok = W.make_tokens(w, B)
    lq_o, pr_o = O.tok_log_prob(w, wt, pe, rp, col, tok)
    lq_g, cp_g = model.log_prob(dev(tok.astype(np.uint8)).view(torch.int8), want_cond_p=True)
    cp_g, lq_g = cp_g.cpu().numpy().astype(np.float64), lq_g.cpu().numpy().astype(np.float64)
    picked = np.take_along_axis(pr_o, tok[..., None], axis=-1)[..., 0]
    assert np.abs(cp_g - picked).max() <= TOL_P, np.abs(cp_g - picked).max()
    bound = TOL_P * (1.0 / picked).sum(1) + 2.0 * np.spacing(np.abs(lq_o).astype(np.float32)).astype(np.float64)
    assert (np.abs(lq_g - lq_o) <= bound).all()
    # ---- sampling ----
    u = inp["uniforms"]
    tok_g, lq_s, cp_s = model.sample(dev(u), want_cond_p=True)
    tok_g = tok_g.view(torch.uint8).cpu().numpy().astype(np.int32)
    assert tok_g.min() >= 0 and tok_g.max() < V
    lq_o, pr_o = O.tok_log_prob(w, wt, pe, rp, col, tok_g)                  # re-synchronised on the GPU's tokens
    cdf = np.cumsum(pr_o, axis=-1)
    uu = u.astype(np.float64)
    want = np.minimum((uu[..., None] >= cdf).sum(-1), V - 1)
    # the GPU's token k is acceptable iff u lies in the oracle's interval [cdf_{k-1}, cdf_k) widened by the tolerance
    hi = np.take_along_axis(cdf, tok_g[..., None], axis=-1)[..., 0]
    lo = hi - np.take_along_axis(pr_o, tok_g[..., None], axis=-1)[..., 0]
    hi = np.where(tok_g == V - 1, 2.0, hi)                                   # the last token also takes u above the total
    tie = (np.abs(uu - lo) < TOL_P) | (np.abs(uu - hi) < TOL_P)              # u near a boundary of the drawn token's interval
    mism = tok_g != want
    assert ((uu >= lo - TOL_P) & (uu < hi + TOL_P)).all(), "a drawn token whose CDF interval does not contain u"
    assert not (mism & ~tie).any(), f"{(mism & ~tie).sum()} tokens off outside the tie band"
    picked = np.take_along_axis(pr_o, tok_g[..., None], axis=-1)[..., 0]
    assert np.abs(cp_s.cpu().numpy().astype(np.float64) - picked).max() <= TOL_P
    bound = TOL_P * (1.0 / picked).sum(1) + 2.0 * np.spacing(np.abs(lq_o).astype(np.float32)).astype(np.float64)
    assert (np.abs(lq_s.cpu().numpy().astype(np.float64) - lq_o) <= bound).all()
    # chain rule on the GPU, and determinism
    lq_tf, cp_tf = model.log_prob(dev(tok_g.astype(np.uint8)).view(torch.int8), want_cond_p=True)
    assert (cp_tf - cp_s).abs().max().item() <= 2e-4
    assert (lq_tf - lq_s).abs().max().item() <= 2e-4 * max(1.0, lq_s.abs().max().item())
    again = model.sample(dev(u), want_cond_p=True)
    assert torch.equal(again[0].view(torch.uint8).cpu(), torch.from_numpy(tok_g.astype(np.uint8)))
    print(f"{case}: V={V}, {w.n_sites} tokens, near-boundary sites {int(tie.sum())} of {tie.size}, "
          f"tokens off among them {int(mism.sum())}, distinct tokens drawn {len(np.unique(tok_g))}")
    # ---- tokens -> lattice spins -> energy ----
    si = inp["site_index"]
    s_g = fv.tokens_to_spins(dev(tok_g.astype(np.uint8)), dev(si))
    s_o = O.tokens_to_spins(tok_g, si)
    assert np.array_equal(s_g.cpu().numpy(), s_o)
    E_g = fv.energy_csr(s_g, dev(inp["bond_rowptr"]), dev(inp["bond_col"]), dev(inp["bond_val"]), base.coupling == "pm1")
    E_o = O.energy_csr(s_o, inp["bond_rowptr"], inp["bond_col"], inp["bond_val"])
    if base.coupling == "pm1":
        assert np.array_equal(E_g.cpu().numpy().astype(np.float64), E_o)
    else:
        scale = np.maximum(np.abs(E_o), np.sqrt((inp["bond_val"].astype(np.float64) ** 2).sum()))
        assert (np.abs(E_g.cpu().numpy() - E_o) <= 1e-4 * scale).all()
    model.close()


def test_patch_tokens_shape_errors():
    w = W.patched(dataclasses.replace(W.CONFIGS["cfg2"], L=8, n_sites=64, window=2))
    inp = W.make_all(w, batch=4)
    bad = dataclasses.replace(w, vocab=5)
    with pytest.raises(fv.FlashVanError):
        fv.create_model(bad, inp["weights"], inp["mask_rowptr"], inp["mask_col"], inp["posemb"], 4)
    with pytest.raises(fv.FlashVanError):                                   # W_O is not part of the patched path
        fv.create_model(dataclasses.replace(w, has_wo=1), inp["weights"], inp["mask_rowptr"], inp["mask_col"], inp["posemb"], 4)
