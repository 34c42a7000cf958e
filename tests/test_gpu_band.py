"""GPU parity of the band-only fast path (Eq. S1: M_ij = 0 iff i - j <= W).

When every mask row is the one run max(0, t-W)..t, fv_create_model gives fv_sample a ring-buffer KV window of W+1 rows
per (sample, layer).  Checked here: the detection (kv_window / kv_bytes), sample and log_prob against the fp64 oracle
under the band mask, and that the window changes nothing -- the same uniforms through the N-row pool
(FLASHVAN_KV=dense) give bit-identical spins, log q and conditionals -- for the three samplers.
"""
import dataclasses

import numpy as np
import pytest
import torch

from paper_2606_22984_b200 import binding as fv
from paper_2606_22984_b200 import workloads as W
from test_gpu_parity import build, check_log_prob, check_sample, dev

pytestmark = pytest.mark.gpu


def band_workload(base, N, **kw):
    return dataclasses.replace(W.CONFIGS[base], L=N, n_sites=N, **kw)


# (base config, N, W, B): widths below, at and above a ring chunk (16 rows), a window that does not divide N,
# one sample per CTA up to several n8-tiles per CTA, W + 1 = N / 2 exactly (largest window taken)
CASES = [("cfg5", 150, 12, 19), ("cfg5", 200, 16, 150), ("cfg5", 257, 37, 300), ("cfg2", 96, 5, 75),
         ("cfg4", 130, 64, 41), ("cfg3", 64, 1, 9), ("cfg1", 40, 19, 33)]


@pytest.mark.parametrize("base,N,width,B", CASES)
def test_band_window_against_oracle_and_dense_pool(base, N, width, B, monkeypatch):
    w = band_workload(base, N, n_layers=min(W.CONFIGS[base].n_layers, 3))
    mask = W.band_mask_csr(N, width)
    model, weights, posemb, rp, col = build(w, B, mask=mask)
    assert model.kv_window == width + 1
    assert model.kv_bytes == B * w.n_layers * (width + 1) * 2 * w.d_model * 2
    check_log_prob(w, model, weights, posemb, rp, col, W.make_spins(w, B, seed=width))
    u = W.make_uniforms(w, B, seed=width)
    ties, flips = check_sample(w, model, weights, posemb, rp, col, u)
    print(f"band N={N} W={width} B={B}: window {model.kv_window} rows, near-tie sites {ties}, flips among them {flips}")
    got = [x.clone() for x in model.sample(dev(u), want_cond_p=True)]
    again = model.sample(dev(u), want_cond_p=True)                    # a second pass over a used window
    assert all(torch.equal(x, y) for x, y in zip(got, again))
    model.close()
    monkeypatch.setenv("FLASHVAN_KV", "dense")
    dense, *_ = build(w, B, mask=mask)
    assert dense.kv_window == 0 and dense.kv_bytes == B * w.n_layers * N * 2 * w.d_model * 2
    ref = dense.sample(dev(u), want_cond_p=True)
    assert all(torch.equal(x, y) for x, y in zip(got, ref)), "window and N-row pool differ"
    dense.close()


def test_window_is_only_taken_for_pure_bands():
    w = band_workload("cfg5", 96, n_layers=1)
    wts, pe = W.make_weights(w), W.make_posemb(w)
    rp, col = W.band_mask_csr(96, 60)                                  # 2 (W + 1) > N: no gain, N-row pool
    m = fv.create_model(w, wts, rp, col, pe, 4)
    assert m.kv_window == 0
    m.close()
    rp, col = W.band_mask_csr(96, 10)
    rows = [col[rp[t]:rp[t + 1]] for t in range(96)]
    rows[50] = np.concatenate([[3], rows[50]]).astype(np.int32)        # one far key: two runs in row 50
    rp2 = np.concatenate([[0], np.cumsum([len(r) for r in rows])]).astype(np.int32)
    m = fv.create_model(w, wts, rp2, np.concatenate(rows).astype(np.int32), pe, 4)
    assert m.kv_window == 0
    m.close()
    rows = [col[rp[t]:rp[t + 1]] for t in range(96)]
    rows[70] = rows[70][3:]                                            # one shorter row: not the band of a single W
    rp3 = np.concatenate([[0], np.cumsum([len(r) for r in rows])]).astype(np.int32)
    m = fv.create_model(w, wts, rp3, np.concatenate(rows).astype(np.int32), pe, 4)
    assert m.kv_window == 0
    m.close()
    w2 = dataclasses.replace(W.CONFIGS["cfg2"], L=8, n_sites=64, window=8)   # lattice mask with wrap-around keys
    m, *_ = build(w2, 4)
    assert m.kv_window == 0
    m.close()


@pytest.mark.parametrize("kind,B", [("tc", 300), ("tc", 1185), ("chain", 64)])
def test_band_window_on_the_tcgen05_samplers(kind, B, monkeypatch):
    """The tcgen05 streaming sampler (default from 9 samples per CTA on) and the weight-stationary chain read the
    same copy plan: d = 128, 16-wide heads."""
    N, width = 160, 21
    w = band_workload("cfg5", N, n_layers=3)
    mask = W.band_mask_csr(N, width)
    monkeypatch.setenv("FLASHVAN_DECODE", kind)
    model, weights, posemb, rp, col = build(w, B, mask=mask)
    assert model.kv_window == width + 1
    assert model.sampler_kind(B) == ("ring-tc" if kind == "tc" else "chain")
    u = W.make_uniforms(w, B, seed=3)
    check_sample(w, model, weights, posemb, rp, col, u)
    got = [x.clone() for x in model.sample(dev(u), want_cond_p=True)]
    model.close()
    monkeypatch.setenv("FLASHVAN_KV", "dense")
    dense, *_ = build(w, B, mask=mask)
    ref = dense.sample(dev(u), want_cond_p=True)
    assert all(torch.equal(x, y) for x, y in zip(got, ref))
    dense.close()
