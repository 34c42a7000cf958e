"""Oracle for the ordered Markov boundary (TEST INFRASTRUCTURE ONLY -- only tests/ may import this).

PAPER.md:256-273 (Sec. IV.A.1, Eq. 12-13): for an Ising model on a graph G = (V, E) with the vertices
numbered in sampling order, the ordered Markov boundary of vertex i is the set of past vertices j < i
that are adjacent to i, or joined to i by a path j -> v_1 -> ... -> v_k -> i whose intermediate vertices
all lie in the future (v > i).  PAPER.md:549-557 (SI I.A, Eq. S1) turns it into the attention mask: a
sliding window of width W >= d_max = max_{j in boundary(i)} (i - j).

The functions below are that definition written out (one graph search per vertex, nothing shared
between vertices) plus, for the pins, the conditional independence statement of Eq. 12 checked by exact
enumeration of the Boltzmann distribution.  Pins: tests/test_markov.py.
"""
import itertools

import numpy as np


def ordered_markov_boundary(n, edges):
    """boundary[i] = sorted list of j < i adjacent to i or reachable from i through vertices > i only.

    `edges` is any iterable of pairs (a, b), a != b, vertices already numbered in sampling order."""
    nbr = [set() for _ in range(n)]
    for a, b in edges:
        a, b = int(a), int(b)
        if a == b:
            raise ValueError("self loop")
        nbr[a].add(b)
        nbr[b].add(a)
    out = []
    for i in range(n):
        found = set()
        seen = {i}
        stack = [i]
        while stack:                      # walk from i; only future vertices are walked through
            v = stack.pop()
            for u in nbr[v]:
                if u < i:
                    found.add(u)          # a past vertex ends the path
                elif u not in seen:
                    seen.add(u)
                    stack.append(u)
        out.append(sorted(found))
    return out


def d_max(boundary):
    """d_max = max_i max_{j in boundary(i)} (i - j); 0 for a graph without edges."""
    return max([i - j for i, b in enumerate(boundary) for j in b], default=0)


def boundary_to_mask_csr(boundary):
    """Position-space attention rows (DESIGN.md reading: position t carries spin t-1, position 0 the start
    token, a row always holds its own position): row t = {j + 1 : j in boundary(t)} U {t}."""
    rowptr = np.zeros(len(boundary) + 1, dtype=np.int32)
    cols = []
    for t, b in enumerate(boundary):
        cols.extend(sorted({j + 1 for j in b} | {t}))
        rowptr[t + 1] = len(cols)
    return rowptr, np.asarray(cols, dtype=np.int32)


def conditional_dependence_set(n, J, i, beta=1.0, tol=1e-12):
    """Eq. 12-13 by brute force: the set of past vertices j < i on which P(s_i = +1 | s_0..s_{i-1}) of the
    Boltzmann distribution exp(beta * sum_{a<b} J_ab s_a s_b) actually depends (flipping s_j changes it
    for at least one setting of the other past spins).  Only for tiny n."""
    J = np.asarray(J, dtype=np.float64)
    states = np.array(list(itertools.product((-1.0, 1.0), repeat=n)))
    energy = -0.5 * np.einsum("sa,ab,sb->s", states, J, states)
    weight = np.exp(-beta * energy)

    def p_up(past):
        sel = np.all(states[:, :i] == np.asarray(past), axis=1) if i else np.ones(len(states), bool)
        up = sel & (states[:, i] > 0)
        return weight[up].sum() / weight[sel].sum()

    dep = set()
    for past in itertools.product((-1.0, 1.0), repeat=i):
        base = p_up(past)
        for j in range(i):
            flipped = list(past)
            flipped[j] = -flipped[j]
            if abs(p_up(flipped) - base) > tol:
                dep.add(j)
    return sorted(dep)


def lattice_edges(L, dim, periodic):
    """Nearest-neighbour edges of the L^dim hypercubic lattice in raster order (last axis fastest)."""
    strides = [L ** (dim - 1 - a) for a in range(dim)]
    edges = set()
    for c in itertools.product(range(L), repeat=dim):
        i = sum(c[a] * strides[a] for a in range(dim))
        for a in range(dim):
            if c[a] + 1 < L or (periodic and L > 2):
                d = list(c)
                d[a] = (c[a] + 1) % L
                j = sum(d[b] * strides[b] for b in range(dim))
                edges.add((min(i, j), max(i, j)))
    return sorted(edges)
