"""Ordered Markov boundary: pins of the oracle, then the library's host-side
builder `fv_markov_mask` against the oracle, bit-exact.  No GPU needed (host logic only)."""
import itertools

import numpy as np
import pytest

from oracle import markov as OM


# ------------------------------------------------------------------ pins of the oracle

def _random_graph(rng, n, p):
    return [(a, b) for a in range(n) for b in range(a + 1, n) if rng.random() < p]


@pytest.mark.parametrize("seed", range(6))
def test_oracle_boundary_is_the_exact_conditioning_set(seed):
    """Eq. 12: with generic couplings P(s_i | past) depends on exactly the boundary (brute force over all
    2^n states; the path characterisation is never used on the brute-force side)."""
    rng = np.random.default_rng(100 + seed)
    n = 7
    edges = _random_graph(rng, n, 0.35)
    J = np.zeros((n, n))
    for a, b in edges:
        J[a, b] = J[b, a] = rng.normal()
    boundary = OM.ordered_markov_boundary(n, edges)
    for i in range(n):
        assert OM.conditional_dependence_set(n, J, i) == boundary[i], (i, edges)


def test_oracle_conditioning_set_on_a_small_open_lattice():
    L = 3
    edges = OM.lattice_edges(L, 2, periodic=False)
    rng = np.random.default_rng(7)
    J = np.zeros((9, 9))
    for a, b in edges:
        J[a, b] = J[b, a] = rng.choice([-1.0, 1.0]) * (0.5 + rng.random())
    boundary = OM.ordered_markov_boundary(9, edges)
    for i in range(9):
        assert OM.conditional_dependence_set(9, J, i, beta=0.7) == boundary[i]


@pytest.mark.parametrize("L", [2, 3, 5, 8])
def test_oracle_open_2d_raster_is_the_previous_L_spins(L):
    """the 2D cut is the current row so far plus the rest of the previous row.  In the last
    row nothing unsampled is left below, so only the neighbours and the part of the previous row that
    still touches unsampled sites remain."""
    boundary = OM.ordered_markov_boundary(L * L, OM.lattice_edges(L, 2, periodic=False))
    for i in range(L * L):
        r, c = divmod(i, L)
        if r < L - 1:
            assert boundary[i] == list(range(max(0, i - L), i))
        else:
            assert boundary[i] == sorted(set(range(i - L, i - c)) | ({i - 1} if c else set()))
    assert OM.d_max(boundary) == L


def test_oracle_periodic_2d_boundary_is_at_most_2L():
    """Periodic rows and columns: the first row stays on the frontier until the last row is sampled, so the
    boundary is the previous L spins plus the first row (and the row's own first site): |boundary| <= 2L."""
    L = 8
    boundary = OM.ordered_markov_boundary(L * L, OM.lattice_edges(L, 2, periodic=True))
    assert max(len(b) for b in boundary) == 2 * L
    edges = set(OM.lattice_edges(L, 2, periodic=True))
    for i in range(L * L):
        r, c = divmod(i, L)
        if r < L - 1:
            want = set(range(max(0, i - L), i))         # the open-lattice cut
            if r > 0:
                want |= set(range(0, L))                # the first row, seen through the unsampled last row
            if c > 0:
                want.add(r * L)                         # the row's first site, through the periodic row bond
            assert set(boundary[i]) == {j for j in want if j < i}, (i, boundary[i])
        else:                                           # last row: the frontier shrinks as the lattice fills up
            direct = {j for j in range(i) if (j, i) in edges}
            assert direct <= set(boundary[i]) <= set(range(i - L, i)) | set(range(c, L)), (i, boundary[i])


def test_oracle_conditioning_set_on_a_small_periodic_lattice():
    L = 3
    edges = OM.lattice_edges(L, 2, periodic=True)
    assert len(edges) == 18
    rng = np.random.default_rng(11)
    J = np.zeros((9, 9))
    for a, b in edges:
        J[a, b] = J[b, a] = rng.normal()
    boundary = OM.ordered_markov_boundary(9, edges)
    for i in range(9):
        assert OM.conditional_dependence_set(9, J, i, beta=0.6) == boundary[i]


def test_oracle_chain_complete_and_empty_graphs():
    n = 9
    chain = OM.ordered_markov_boundary(n, [(i, i + 1) for i in range(n - 1)])
    assert chain == [[]] + [[i - 1] for i in range(1, n)] and OM.d_max(chain) == 1      # PAPER.md:549, 1D
    full = OM.ordered_markov_boundary(n, itertools.combinations(range(n), 2))
    assert full == [list(range(i)) for i in range(n)]                                   # SK: whole past
    assert OM.ordered_markov_boundary(4, []) == [[], [], [], []]
    # a path through the future: 0 - 3 - 1, vertex 2 isolated
    assert OM.ordered_markov_boundary(4, [(0, 3), (1, 3)]) == [[], [0], [], [0, 1]]


def test_oracle_open_3d_window():
    """d_max = O(L^2) in 3D; open raster gives exactly the previous L^2 spins."""
    L = 3
    boundary = OM.ordered_markov_boundary(L ** 3, OM.lattice_edges(L, 3, periodic=False))
    for i in range((L - 1) * L * L):                   # every layer but the last (nothing unsampled beyond it)
        assert boundary[i] == list(range(max(0, i - L * L), i))
    assert OM.d_max(boundary) == L * L


def test_oracle_mask_rows():
    rowptr, col = OM.boundary_to_mask_csr([[], [0], [], [0, 1]])
    assert rowptr.tolist() == [0, 1, 2, 3, 6] and col.tolist() == [0, 1, 2, 1, 2, 3]


# ------------------------------------------------------------------ the library's builder against the oracle

def _lib_rows(n, edges, position_space):
    from paper_2606_22984_b200 import binding as fv
    from paper_2606_22984_b200 import build as fvbuild
    fvbuild.build()
    e = np.asarray(list(edges), dtype=np.int32).reshape(-1, 2)
    return fv.markov_mask(n, e[:, 0], e[:, 1], position_space)


def _oracle_csr(boundary):
    rowptr = np.cumsum([0] + [len(b) for b in boundary]).astype(np.int32)
    col = np.asarray([j for b in boundary for j in b], dtype=np.int32)
    return rowptr, col


CASES = [("open2d_L8", 64, OM.lattice_edges(8, 2, False)),
         ("periodic2d_L8", 64, OM.lattice_edges(8, 2, True)),
         ("periodic2d_L16", 256, OM.lattice_edges(16, 2, True)),
         ("open3d_L4", 64, OM.lattice_edges(4, 3, False)),
         ("periodic3d_L4", 64, OM.lattice_edges(4, 3, True)),
         ("chain", 17, [(i, i + 1) for i in range(16)]),
         ("complete", 33, list(itertools.combinations(range(33), 2))),
         ("no_edges", 5, []),
         ("single_vertex", 1, [])]


@pytest.mark.parametrize("name,n,edges", CASES, ids=[c[0] for c in CASES])
def test_library_matches_oracle(name, n, edges):
    boundary = OM.ordered_markov_boundary(n, edges)
    rowptr, col, dmax = _lib_rows(n, edges, position_space=False)
    want_ptr, want_col = _oracle_csr(boundary)
    assert np.array_equal(rowptr, want_ptr) and np.array_equal(col, want_col)
    assert dmax == OM.d_max(boundary)
    rowptr, col, _ = _lib_rows(n, edges, position_space=True)
    want_ptr, want_col = OM.boundary_to_mask_csr(boundary)
    assert np.array_equal(rowptr, want_ptr) and np.array_equal(col, want_col)


@pytest.mark.parametrize("seed", range(8))
def test_library_matches_oracle_on_random_graphs_and_orderings(seed):
    """Random sparse graphs, a random relabelling of a lattice (a non-raster ordering), duplicate and
    reversed edges."""
    rng = np.random.default_rng(500 + seed)
    n = int(rng.integers(2, 120))
    edges = _random_graph(rng, n, float(rng.choice([0.02, 0.05, 0.2])))
    edges += [(b, a) for a, b in edges[::3]]                         # reversed duplicates
    if seed % 2:
        perm = rng.permutation(64)
        edges = [(int(perm[a]), int(perm[b])) for a, b in OM.lattice_edges(8, 2, True)]
        n = 64
    boundary = OM.ordered_markov_boundary(n, edges)
    rowptr, col, dmax = _lib_rows(n, edges, position_space=False)
    want_ptr, want_col = _oracle_csr(boundary)
    assert np.array_equal(rowptr, want_ptr) and np.array_equal(col, want_col) and dmax == OM.d_max(boundary)


def test_library_mask_is_accepted_shape_for_cfg5_lattice():
    """Full size: 2D periodic L = 64 (the cfg5 lattice).  Properties that hold at any size: rows ascending and
    unique, last entry == t, every direct past neighbour present, |row| <= 2L + 1, window 2L... contains it."""
    L = 64
    edges = OM.lattice_edges(L, 2, True)
    rowptr, col, dmax = _lib_rows(L * L, edges, position_space=True)
    assert rowptr[0] == 0 and rowptr[-1] == len(col)
    assert int(np.diff(rowptr).max()) <= 2 * L + 1
    assert dmax == L * L - L                                     # the first row stays visible up to the last row
    nbr = [[] for _ in range(L * L)]
    for a, b in edges:
        nbr[b].append(a)
    for t in range(L * L):
        row = col[rowptr[t]:rowptr[t + 1]]
        assert row[-1] == t and np.all(np.diff(row) > 0) and row[0] >= 0
        assert all((j + 1 in row) for j in nbr[t] if j < t)
    # sampled rows against the oracle's definition (one graph search each)
    sample = [0, 1, L - 1, L, L + 1, 2 * L + 5, 2000, L * L - L - 1, L * L - L, L * L - 2, L * L - 1]
    nb = [set() for _ in range(L * L)]
    for a, b in edges:
        nb[a].add(b)
        nb[b].add(a)
    for t in sample:
        found, seen, stack = set(), {t}, [t]
        while stack:
            v = stack.pop()
            for u in nb[v]:
                if u < t:
                    found.add(u)
                elif u not in seen:
                    seen.add(u)
                    stack.append(u)
        assert col[rowptr[t]:rowptr[t + 1]].tolist() == sorted({j + 1 for j in found} | {t})


def test_library_rejects_bad_edges():
    from paper_2606_22984_b200 import binding as fv
    with pytest.raises(fv.FlashVanError):
        _lib_rows(4, [(0, 4)], False)
    with pytest.raises(fv.FlashVanError):
        _lib_rows(4, [(2, 2)], False)
