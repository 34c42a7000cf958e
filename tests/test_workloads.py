"""Seeded input generators: mask statistics and rows stated in SURVEY.md 8(d) / DESIGN.md."""
import numpy as np

from paper_2606_22984_b200 import workloads as W


def test_mask_statistics():
    want = {"cfg1": 136, "cfg2": 3070, "cfg3": 131328, "cfg4": 23165, "cfg5": 268385}
    for name, nnz in want.items():
        w = W.CONFIGS[name]
        rp, col = W.make_mask_csr(w)
        assert rp[-1] == nnz == col.size
        for t in range(0, w.n_sites, max(1, w.n_sites // 97)):
            row = col[rp[t]:rp[t + 1]]
            assert row[-1] == t and np.all(np.diff(row) > 0) and row[0] >= 0
    rp, col = W.make_mask_csr(W.CONFIGS["cfg2"])
    assert col[rp[17]:rp[18]].tolist() == [1, 2, 3] + list(range(10, 18))
    assert col[rp[255]:rp[256]].tolist() == [1, 15, 16, 32, 224, 225, 239, 240, 241, 242] + list(range(248, 256))
    assert col[rp[0]:rp[1]].tolist() == [0]


def test_couplings_and_blob():
    for name in ("cfg2", "cfg4", "cfg5"):
        w = W.CONFIGS[name]
        rp, col, val = W.make_couplings_ea(w)
        assert rp[-1] == w.dim * w.n_sites and np.all(col > np.repeat(np.arange(w.n_sites), np.diff(rp)))
        if w.coupling == "pm1":
            assert set(np.unique(val)) == {-1.0, 1.0}
    J = W.make_couplings_sk(W.CONFIGS["cfg3"])
    assert abs(J.var() * 512 - 1.0) < 0.02
    assert W.n_weights(W.CONFIGS["cfg5"]) == 1090822
    u = W.make_uniforms(W.CONFIGS["cfg1"])
    assert u.dtype == np.float32 and u.min() >= 0 and u.max() < 1
    assert np.array_equal(u, W.make_uniforms(W.CONFIGS["cfg1"]))


def test_band_mask():
    rp, col = W.band_mask_csr(10, 3)
    assert col[rp[5]:rp[6]].tolist() == [2, 3, 4, 5] and col[rp[1]:rp[2]].tolist() == [0, 1]
