"""fv_log_prob_static: the teacher-forced pass with its workspace in the library's file-scope `static __device__`
array (no cudaMalloc in the call) against the existing fv_log_prob on the same spins -- same kernels, so the results
must be bit-identical, which is inside every tolerance the parity tests use.  Two calls in a row (the second one finds
the first one's contents in the array), on two models of different shape sharing the array, plus the size limit.
Collected last (file name): pytest -x must not hide other tests behind it."""
import dataclasses

import numpy as np
import pytest
import torch

from paper_2606_22984_b200 import binding as fv
from paper_2606_22984_b200 import workloads as W

pytestmark = pytest.mark.gpu
STATIC_BYTES = 64 << 20


def make(w, B):
    rp, col = W.make_mask_csr(w)
    return fv.create_model(w, W.make_weights(w), rp, col, W.make_posemb(w), B)


def rows_that_fit(w):
    return STATIC_BYTES // (w.d_model * (8 + 4 * w.n_layers))


def test_static_workspace_matches_fv_log_prob_twice_in_a_row():
    w5 = dataclasses.replace(W.CONFIGS["cfg5"], L=16, n_sites=256, window=16)      # 6 layers, d = 128: 4 KB per row
    w2 = dataclasses.replace(W.CONFIGS["cfg2"], L=8, n_sites=64, window=8)         # 4 layers, d = 64
    B5, B2 = 37, 150
    assert B5 * w5.n_sites <= rows_that_fit(w5) and B2 * w2.n_sites <= rows_that_fit(w2)
    m5, m2 = make(w5, B5), make(w2, B2)
    for rep in range(2):
        for model, w, B in ((m5, w5, B5), (m2, w2, B2)):                            # the two models share the array
            spins = torch.from_numpy(W.make_spins(w, B, seed=20 + rep)).cuda()
            lq_ref, cp_ref = model.log_prob(spins, want_cond_p=True)
            lq = torch.full((B,), float("nan"), device="cuda")
            cp = torch.full((B, w.n_sites), float("nan"), device="cuda")
            torch.cuda.synchronize()
            before = torch.cuda.memory_allocated()
            model.log_prob_static(spins, lq, cp)
            assert torch.cuda.memory_allocated() == before
            torch.cuda.synchronize()
            assert torch.isfinite(lq).all() and torch.isfinite(cp).all()
            assert torch.equal(lq, lq_ref) and torch.equal(cp, cp_ref), (rep, w.n_sites, (lq - lq_ref).abs().max().item())
            lq2 = torch.empty_like(lq)                                              # second call, no cond_p
            model.log_prob_static(spins, lq2)
            assert torch.equal(lq2, lq_ref)
    m5.close()
    m2.close()


def test_static_workspace_limit_and_shapes():
    w5 = dataclasses.replace(W.CONFIGS["cfg5"], L=16, n_sites=256, window=16)
    fit = rows_that_fit(w5) // w5.n_sites                                           # 64 samples of 256 sites
    model = make(w5, fit + 1)
    spins = torch.from_numpy(W.make_spins(w5, fit + 1, seed=5)).cuda()
    lq = torch.empty(fit + 1, device="cuda")
    with pytest.raises(fv.FlashVanError, match="static array holds"):
        model.log_prob_static(spins, lq)
    ref, _ = model.log_prob(spins[:fit].contiguous())
    got, _ = model.log_prob_static(spins[:fit].contiguous(), lq[:fit])              # exactly at the limit
    assert torch.equal(got, ref)
    model.close()
    wide = dataclasses.replace(W.CONFIGS["cfg2"], L=6, n_sites=36, window=5, n_layers=2, d_model=256, n_heads=4)
    model = make(wide, 4)                                                           # d = 256 has no layer-major path
    with pytest.raises(fv.FlashVanError, match="layer-major"):
        model.log_prob_static(torch.from_numpy(W.make_spins(wide, 4)).cuda(), torch.empty(4, device="cuda"))
    model.close()
    wo = dataclasses.replace(W.CONFIGS["cfg2"], L=6, n_sites=36, window=5, n_layers=2, has_wo=1)
    model = make(wo, 4)                                                             # W_O: the extra tcgen05 GEMM per layer
    spins = torch.from_numpy(W.make_spins(wo, 4)).cuda()
    ref, _ = model.log_prob(spins)
    got, _ = model.log_prob_static(spins, torch.empty(4, device="cuda"))
    assert torch.equal(got, ref)
    model.close()
