"""Replica overlap q = sigma^1 . sigma^2 / N (Eq. 9): pins of the oracle (no GPU)."""
import numpy as np

from oracle import oracle as O


def _spins(rng, B, N):
    return (rng.integers(0, 2, size=(B, N)) * 2 - 1).astype(np.int8)


def test_overlap_closed_forms():
    rng = np.random.default_rng(3)
    B, N = 37, 101
    a = _spins(rng, B, N)
    dot, hist = O.overlap(a, a)
    assert (dot == N).all() and hist[N] == B and hist.sum() == B            # q = 1 with itself
    dot, hist = O.overlap(a, -a)
    assert (dot == -N).all() and hist[0] == B                               # q = -1 with its mirror image
    # flipping k spins of a copy lowers the sum by 2k: q = 1 - 2k/N
    c = a.copy()
    ks = rng.integers(0, N + 1, size=B)
    for b, k in enumerate(ks):
        c[b, rng.choice(N, size=k, replace=False)] *= -1
    dot, hist = O.overlap(a, c)
    assert (dot == N - 2 * ks).all()
    assert (hist == np.bincount(N - ks, minlength=N + 1)).all()


def test_overlap_symmetries_and_parity():
    rng = np.random.default_rng(4)
    B, N = 64, 50
    a, c = _spins(rng, B, N), _spins(rng, B, N)
    dot, hist = O.overlap(a, c)
    assert ((dot + N) % 2 == 0).all() and (np.abs(dot) <= N).all() and hist.sum() == B
    assert (O.overlap(c, a)[0] == dot).all()                                 # symmetric
    assert (O.overlap(-a, c)[0] == -dot).all() and (O.overlap(-a, -c)[0] == dot).all()
    assert (O.overlap(-a, c)[1] == hist[::-1]).all()                         # p(q) -> p(-q)
    assert (dot == np.einsum("bi,bi->b", a.astype(np.int64), c.astype(np.int64))).all()
    # a gauge transformation of both replicas leaves q alone
    g = _spins(rng, 1, N)
    assert (O.overlap(a * g, c * g)[0] == dot).all()


def test_overlap_of_independent_uniform_spins_has_variance_one_over_N():
    rng = np.random.default_rng(5)
    B, N = 20000, 64
    dot, _ = O.overlap(_spins(rng, B, N), _spins(rng, B, N))
    q = dot / N
    assert abs(q.mean()) < 5 / np.sqrt(B * N) and abs(q.var() * N - 1) < 0.05
