"""ctypes wrapper around oracle/flashvan_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It shares nothing with paper_2606_22984_b200/ except that both are
handed the arrays produced by paper_2606_22984_b200/workloads.py (seeded inputs only).

Every function takes the *host numpy arrays* of the workload and returns fp64 results.
Citations are in flashvan_oracle.c next to each step.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "flashvan_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


class _Cfg(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in
                ("n_sites", "n_layers", "d_model", "n_heads", "d_token", "ffn_mult",
                 "has_wo", "act", "ln2_style")] + [("ln_eps", ctypes.c_double), ("vocab", ctypes.c_int32)]


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (-O3 -fopenmp); returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-fPIC", "-shared", "-std=c99",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, capture_output=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.fvo_n_weights.restype = ctypes.c_int64
        _lib.fvo_sample.restype = ctypes.c_int
        _lib.fvo_log_prob.restype = ctypes.c_int
        _lib.fvo_tok_sample.restype = ctypes.c_int
        _lib.fvo_tok_log_prob.restype = ctypes.c_int
        _lib.fvo_energy_dense.restype = None
        _lib.fvo_energy_csr.restype = None
    return _lib


def _cfg(w) -> _Cfg:
    return _Cfg(w.n_sites, w.n_layers, w.d_model, w.n_heads, w.d_token, w.ffn_mult,
                w.has_wo, 0, w.ln2_style, float(w.ln_eps), int(getattr(w, "vocab", 2)))


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _c(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def n_threads() -> int:
    """Threads the OpenMP runtime will use (OMP_NUM_THREADS or all cores)."""
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else (os.cpu_count() or 1)


def n_weights(w) -> int:
    return int(_load().fvo_n_weights(ctypes.byref(_cfg(w))))


def sample(w, weights, posemb, rowptr, col, uniforms):
    """Alg. 2.  Returns spins int8 [B,N], logq f64 [B], cond_p f64 [B,N]."""
    lib = _load()
    weights, posemb = _c(weights, np.float32), _c(posemb, np.float32)
    rowptr, col = _c(rowptr, np.int32), _c(col, np.int32)
    uniforms = _c(uniforms, np.float32)
    assert weights.size == n_weights(w) and posemb.shape == (w.n_sites, w.d_pos)
    B = uniforms.shape[0]
    spins = np.empty((B, w.n_sites), np.int8)
    logq = np.empty(B, np.float64)
    cp = np.empty((B, w.n_sites), np.float64)
    rc = lib.fvo_sample(ctypes.byref(_cfg(w)), _p(weights), _p(posemb), _p(rowptr), _p(col),
                        ctypes.c_int32(B), _p(uniforms), _p(spins), _p(logq), _p(cp))
    if rc != 0:
        raise MemoryError("oracle sample failed")
    return spins, logq, cp


def log_prob(w, weights, posemb, rowptr, col, spins):
    """Alg. 1.  Returns logq f64 [B], cond_p = p_t(+1) f64 [B,N]."""
    lib = _load()
    weights, posemb = _c(weights, np.float32), _c(posemb, np.float32)
    rowptr, col = _c(rowptr, np.int32), _c(col, np.int32)
    spins = _c(spins, np.int8)
    assert weights.size == n_weights(w) and posemb.shape == (w.n_sites, w.d_pos)
    B = spins.shape[0]
    logq = np.empty(B, np.float64)
    cp = np.empty((B, w.n_sites), np.float64)
    rc = lib.fvo_log_prob(ctypes.byref(_cfg(w)), _p(weights), _p(posemb), _p(rowptr), _p(col),
                          ctypes.c_int32(B), _p(spins), _p(logq), _p(cp))
    if rc != 0:
        raise MemoryError("oracle log_prob failed")
    return logq, cp


def tok_sample(w, weights, posemb, rowptr, col, uniforms):
    """Alg. 2 with patch tokens: inverse-CDF draw of one of w.vocab tokens per position.
    Returns tokens int32 [B,N], logq f64 [B], probs f64 [B,N,V] (the full conditional of every position)."""
    lib = _load()
    weights, posemb = _c(weights, np.float32), _c(posemb, np.float32)
    rowptr, col = _c(rowptr, np.int32), _c(col, np.int32)
    uniforms = _c(uniforms, np.float32)
    assert weights.size == n_weights(w) and posemb.shape == (w.n_sites, w.d_pos)
    B = uniforms.shape[0]
    tokens = np.empty((B, w.n_sites), np.int32)
    logq = np.empty(B, np.float64)
    probs = np.empty((B, w.n_sites, w.vocab), np.float64)
    rc = lib.fvo_tok_sample(ctypes.byref(_cfg(w)), _p(weights), _p(posemb), _p(rowptr), _p(col),
                            ctypes.c_int32(B), _p(uniforms), _p(tokens), _p(logq), _p(probs))
    if rc != 0:
        raise MemoryError("oracle tok_sample failed")
    return tokens, logq, probs


def tok_log_prob(w, weights, posemb, rowptr, col, tokens):
    """Alg. 1 with patch tokens: log q of given token sequences and the full conditionals [B,N,V]."""
    lib = _load()
    weights, posemb = _c(weights, np.float32), _c(posemb, np.float32)
    rowptr, col = _c(rowptr, np.int32), _c(col, np.int32)
    tokens = _c(tokens, np.int32)
    assert weights.size == n_weights(w) and posemb.shape == (w.n_sites, w.d_pos)
    assert tokens.min() >= 0 and tokens.max() < w.vocab
    B = tokens.shape[0]
    logq = np.empty(B, np.float64)
    probs = np.empty((B, w.n_sites, w.vocab), np.float64)
    rc = lib.fvo_tok_log_prob(ctypes.byref(_cfg(w)), _p(weights), _p(posemb), _p(rowptr), _p(col),
                              ctypes.c_int32(B), _p(tokens), _p(logq), _p(probs))
    if rc != 0:
        raise MemoryError("oracle tok_log_prob failed")
    return logq, probs


def tokens_to_spins(tokens, site_index):
    """Unpack patch tokens into lattice spins: bit k of token n is the spin of lattice site site_index[n, k]
    (the index list comes from workloads.patch_site_index), spin = 2 bit - 1."""
    tokens = np.asarray(tokens, np.int64)
    B, n_tok = tokens.shape
    P = site_index.shape[1]
    spins = np.zeros((B, n_tok * P), np.int8)
    for k in range(P):
        spins[:, site_index[:, k]] = (2 * ((tokens >> k) & 1) - 1).astype(np.int8)
    return spins


def energy_dense(spins, J):
    """E = -sum_{i<j} J_ij s_i s_j, explicit double loop (Eq. 6)."""
    spins, J = _c(spins, np.int8), _c(J, np.float32)
    B, N = spins.shape
    E = np.empty(B, np.float64)
    _load().fvo_energy_dense(ctypes.c_int32(B), ctypes.c_int32(N), _p(spins), _p(J), _p(E))
    return E


def energy_csr(spins, rowptr, col, val):
    """E = -sum_bonds J_ij s_i s_j over the bond list (Eq. 8)."""
    spins = _c(spins, np.int8)
    rowptr, col, val = _c(rowptr, np.int32), _c(col, np.int32), _c(val, np.float32)
    B, N = spins.shape
    E = np.empty(B, np.float64)
    _load().fvo_energy_csr(ctypes.c_int32(B), ctypes.c_int32(N), _p(spins), _p(rowptr),
                           _p(col), _p(val), _p(E))
    return E


def free_energy(E, logq, beta):
    """F_q = mean_b(E_b + T log q_b), T = 1/beta (Eq. 5); returns (mean, std)."""
    f = np.asarray(E, np.float64) + np.asarray(logq, np.float64) / beta
    return float(f.mean()), float(f.std())


def overlap(spins_a, spins_b):
    """Replica overlap (Eq. 9): dot_b = sum_i a_bi * c_bi, an explicit loop over sites in exact
    integers; q_b = dot_b / N.  Returns (dot int64 [B], hist int64 [N + 1]) with hist[(dot + N) / 2] counting
    the samples at each of the N + 1 values -N, -N + 2, ..., N the sum can take (p(q) = hist / B)."""
    a, c = _c(spins_a, np.int8), _c(spins_b, np.int8)
    B, N = a.shape
    dot = np.zeros(B, np.int64)
    for i in range(N):
        dot += a[:, i].astype(np.int64) * c[:, i].astype(np.int64)
    hist = np.zeros(N + 1, np.int64)
    for b in range(B):
        hist[(int(dot[b]) + N) // 2] += 1
    return dot, hist


def param_count(vocab, n_seq, d_token, d_model, n_layers, ffn_mult=4, has_wo=0):
    """Parameter inventory (pin P1, Tables 6-7 l.745-771)."""
    d, f = d_model, ffn_mult * d_model
    per = 2 * d + 3 * (d * d + d) + (d * d + d if has_wo else 0) + 2 * d + f * d + f + d * f + d
    return vocab * d_token + n_seq * (d_model - d_token) + n_layers * per + vocab * d + vocab
