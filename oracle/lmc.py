"""Oracle for the local Monte Carlo refinement of samples (TEST INFRASTRUCTURE ONLY -- only tests/ may import this).

PAPER.md:202, 411 and SI I.C (l.583-595) refine the generated configurations with a "short local Monte Carlo
trajectory" before the loss; the paper gives neither the sweep count nor the acceptance rule, so PARITY WITH THE
AUTHORS' PROCEDURE IS UNPINNED.  What is implemented is the textbook choice, stated here step by step:

  one sweep visits the sites in order i = 0 .. N-1; h_i = sum_j J_ij s_j over the neighbours of i in the order
  the adjacency lists them, accumulated in fp32 (s_j = +-1, so every term is exact and only the additions round);
  dE = 2 s_i h_i (flipping s_i changes E = -sum_{i<j} J_ij s_i s_j, Eq. 6/8, by exactly this); the flip is
  accepted iff beta * dE < e_i, where e_i >= 0 is a caller-supplied standard exponential variate (= -ln u):
  P(accept) = min(1, exp(-beta dE)), the Metropolis rule, with no transcendental inside the sweep, so the
  decision is taken in fp32 from one multiplication and one comparison and can be reproduced bit for bit.

Pins: tests/test_lmc.py (energy bookkeeping against the independent energy routine, beta = 0 and e = 0 closed
forms, the exact one-sweep transition matrix on a 4-site model).
"""
import numpy as np


def sweeps(spins, rowptr, col, val, beta, exp_variates):
    """spins int8 [B, N] (copied), full symmetric adjacency CSR (rowptr[N+1], col, val fp32),
    exp_variates fp32 [B, n_sweeps, N].  Returns (new spins int8 [B, N], accepted flips int64 [B])."""
    s = np.array(spins, dtype=np.int8, copy=True)
    rowptr = np.asarray(rowptr, dtype=np.int64)
    col = np.asarray(col, dtype=np.int64)
    val = np.asarray(val, dtype=np.float32)
    ev = np.asarray(exp_variates, dtype=np.float32)
    B, N = s.shape
    beta32 = np.float32(beta)
    two = np.float32(2.0)
    acc = np.zeros(B, np.int64)
    for b in range(B):
        for k in range(ev.shape[1]):
            for i in range(N):
                h = np.float32(0.0)
                for e in range(rowptr[i], rowptr[i + 1]):
                    h = np.float32(h + val[e] * np.float32(s[b, col[e]]))
                dE = np.float32(two * np.float32(s[b, i]) * h)       # 2 s_i h_i: exact scalings of h
                if np.float32(beta32 * dE) < ev[b, k, i]:
                    s[b, i] = -s[b, i]
                    acc[b] += 1
    return s, acc


def full_adjacency(n, bond_rowptr, bond_col, bond_val):
    """Upper-triangular bond CSR (the energy routines' input) -> full symmetric adjacency CSR, neighbours of a
    site in ascending index order."""
    nb = [[] for _ in range(n)]
    for i in range(n):
        for e in range(bond_rowptr[i], bond_rowptr[i + 1]):
            j = int(bond_col[e])
            nb[i].append((j, float(bond_val[e])))
            nb[j].append((i, float(bond_val[e])))
    rowptr = np.zeros(n + 1, np.int32)
    col, val = [], []
    for i in range(n):
        for j, v in sorted(nb[i]):
            col.append(j)
            val.append(v)
        rowptr[i + 1] = len(col)
    return rowptr, np.asarray(col, np.int32), np.asarray(val, np.float32)
