"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module is the ONLY code shared by the CUDA path and the oracle.  It holds no
arithmetic of the method (no LayerNorm, attention, softmax, energy ...): it only draws
arrays from numpy's PCG64 generator and builds index lists.  Recipe: SURVEY.md §8(d) /
DESIGN.md "Input recipe".

Conventions (readings A3, A11, A12):
  * raster order, last coordinate fastest: i = (z*L + y)*L + x
  * mask CSR is in POSITION space.  Position t's input is the token of spin t-1 (start
    token for t = 0) and its output is the conditional of spin t (Alg. 2).
    A spin-space set S_t ("spin t may see spin j") maps to key positions
    {j+1 : j in S_t} U {t}; rows ascending, unique, last entry = t.
  * couplings: SK  J_ij ~ N(0, 1/N) (variance), symmetric, zero diagonal (Eq. 6
    with the 1/sqrt(N) folded in); EA bonds (i, i+e_axis mod L) listed once, upper-triangular
    CSR (Eq. 8).
"""
from __future__ import annotations

import dataclasses
import itertools
from typing import Optional

import numpy as np


@dataclasses.dataclass(frozen=True)
class Workload:
    name: str
    model: str            # "sk" | "ea"
    dim: int              # lattice dimension (0 for SK)
    L: int                # linear size (N for SK)
    n_sites: int
    n_layers: int
    d_model: int
    n_heads: int
    batch: int
    coupling: str         # "gauss" | "pm1"
    window: int           # previous-W sites in the mask (0 = full causal)
    betas: tuple = (1.0,)
    d_token: int = 2
    ffn_mult: int = 4
    has_wo: int = 0
    ln2_style: int = 0
    ln_eps: float = 1e-5
    vocab: int = 2        # tokens; 2^(patch^dim) when a token stands for a patch of spins
    patch: int = 1        # linear patch size: the model's lattice (L, n_sites) is then the lattice of PATCHES

    @property
    def d_pos(self) -> int:
        return self.d_model - self.d_token

    @property
    def spins_per_token(self) -> int:
        return self.patch ** self.dim if self.patch > 1 else 1


CONFIGS = {
    "cfg1": Workload("cfg1", "sk", 0, 16, 16, 2, 32, 2, 1024, "gauss", 0),
    "cfg2": Workload("cfg2", "ea", 2, 16, 256, 4, 64, 4, 4096, "pm1", 8),
    "cfg3": Workload("cfg3", "sk", 0, 512, 512, 4, 128, 8, 8192, "gauss", 0, betas=(0.5, 1.5)),
    "cfg4": Workload("cfg4", "ea", 3, 10, 1000, 4, 128, 8, 4096, "gauss", 16),
    "cfg5": Workload("cfg5", "ea", 2, 64, 4096, 6, 128, 8, 1024, "pm1", 64),
}

SEED_J, SEED_U, SEED_W, SEED_POS = 0, 1, 2, 3


def small_variant(w: Workload, **kw) -> Workload:
    """A reduced copy of a workload (same laws, smaller sizes) for parity tests."""
    return dataclasses.replace(w, **kw)


# ----------------------------------------------------------------------------- weights
def weight_segments(w: Workload):
    """Ordered (name, shape) list of the fp32 weights blob (SURVEY.md §8(c-2) layout).

    Matrices are row-major [out, in] (y = W x + b, Eq. 2)."""
    d, f = w.d_model, w.ffn_mult * w.d_model
    segs = [("tok_emb", (w.vocab, w.d_token))]
    for l in range(w.n_layers):
        p = f"l{l}."
        segs += [(p + "ln1_g", (d,)), (p + "ln1_b", (d,)),
                 (p + "wq", (d, d)), (p + "bq", (d,)),
                 (p + "wk", (d, d)), (p + "bk", (d,)),
                 (p + "wv", (d, d)), (p + "bv", (d,))]
        if w.has_wo:
            segs += [(p + "wo", (d, d)), (p + "bo", (d,))]
        segs += [(p + "ln2_g", (d,)), (p + "ln2_b", (d,)),
                 (p + "w1", (f, d)), (p + "b1", (f,)),
                 (p + "w2", (d, f)), (p + "b2", (d,))]
    segs += [("head_w", (w.vocab, d)), ("head_b", (w.vocab,))]
    return segs


def n_weights(w: Workload) -> int:
    return int(sum(int(np.prod(s)) for _, s in weight_segments(w)))


def weight_views(w: Workload, blob: np.ndarray) -> dict:
    """Named views into a flat blob (no copies)."""
    out, off = {}, 0
    for name, shape in weight_segments(w):
        n = int(np.prod(shape))
        out[name] = blob[off:off + n].reshape(shape)
        off += n
    assert off == blob.size, (off, blob.size)
    return out


def make_weights(w: Workload, seed: int = SEED_W, std: float = 0.02,
                 head_scale: float = 1.0) -> np.ndarray:
    """normal(0, std) for every entry; LayerNorm gains get +1 (reading A16)."""
    rng = np.random.default_rng(seed)
    blob = rng.normal(0.0, std, size=n_weights(w)).astype(np.float32)
    v = weight_views(w, blob)
    for name in v:
        if name.endswith("ln1_g") or name.endswith("ln2_g"):
            v[name] += np.float32(1.0)
    if head_scale != 1.0:
        v["head_w"] *= np.float32(head_scale)
        v["head_b"] *= np.float32(head_scale)
    return blob


def make_posemb(w: Workload, seed: int = SEED_POS, std: float = 0.02) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return rng.normal(0.0, std, size=(w.n_sites, w.d_pos)).astype(np.float32)


def make_uniforms(w: Workload, batch: Optional[int] = None, seed: int = SEED_U) -> np.ndarray:
    rng = np.random.default_rng(seed)
    b = w.batch if batch is None else batch
    return rng.random(size=(b, w.n_sites), dtype=np.float32)


def make_spins(w: Workload, batch: int, seed: int = 11) -> np.ndarray:
    """Uniform random +-1 configurations (teacher-forced inputs for tests)."""
    rng = np.random.default_rng(seed)
    return (2 * rng.integers(0, 2, size=(batch, w.n_sites)) - 1).astype(np.int8)


def make_tokens(w: Workload, batch: int, seed: int = 11) -> np.ndarray:
    """Uniform random token ids in [0, vocab) (teacher-forced inputs of a patched model)."""
    rng = np.random.default_rng(seed)
    return rng.integers(0, w.vocab, size=(batch, w.n_sites)).astype(np.int32)


# ------------------------------------------------------------------------------ patches
def patched(w: Workload, patch: int = 2) -> Workload:
    """The patched model of an EA workload: one token per patch^dim block of spins, so the
    model's lattice is the lattice of patches (L / patch per side) and the vocabulary has 2^(patch^dim) tokens."""
    assert w.model == "ea" and w.patch == 1 and w.L % patch == 0
    Lt = w.L // patch
    return dataclasses.replace(w, L=Lt, n_sites=Lt ** w.dim, patch=patch, vocab=2 ** (patch ** w.dim))


def spin_lattice(w: Workload) -> Workload:
    """The lattice of SPINS under a patched model (couplings and energies live there)."""
    if w.patch == 1:
        return w
    Ls = w.L * w.patch
    return dataclasses.replace(w, L=Ls, n_sites=Ls ** w.dim, patch=1, vocab=2)


def patch_site_index(w: Workload) -> np.ndarray:
    """[n_tokens, patch^dim] int32: the lattice site (raster index on the spin lattice) whose spin is bit k of
    token n.  Tokens in raster order of the patch lattice; inside a patch the offsets in raster order as well
    (last coordinate fastest), bit 0 = the patch's first site."""
    assert w.patch > 1
    D, p, Lt, Ls = w.dim, w.patch, w.L, w.L * w.patch
    out = np.zeros((w.n_sites, p ** D), dtype=np.int32)
    for n, tc in enumerate(itertools.product(range(Lt), repeat=D)):
        for k, oc in enumerate(itertools.product(range(p), repeat=D)):
            site = 0
            for a in range(D):
                site = site * Ls + tc[a] * p + oc[a]
            out[n, k] = site
    return out


# --------------------------------------------------------------------------- couplings
def site_coords(w: Workload) -> np.ndarray:
    """[N, dim] integer coordinates, most-significant first (z, y, x); x is fastest."""
    assert w.model == "ea"
    idx = np.arange(w.n_sites)
    cols = []
    for a in range(w.dim):
        cols.append((idx // (w.L ** (w.dim - 1 - a))) % w.L)
    return np.stack(cols, axis=1)


def make_couplings_sk(w: Workload, seed: int = SEED_J) -> np.ndarray:
    """Dense symmetric J [N, N] fp32, zero diagonal; upper triangle i<j row-major ~ N(0, 1/N)."""
    assert w.model == "sk"
    n = w.n_sites
    rng = np.random.default_rng(seed)
    iu = np.triu_indices(n, k=1)
    vals = rng.normal(0.0, 1.0 / np.sqrt(n), size=iu[0].size).astype(np.float32)
    J = np.zeros((n, n), dtype=np.float32)
    J[iu] = vals
    J = J + J.T
    return J


def make_couplings_ea(w: Workload, seed: int = SEED_J):
    """Upper-triangular CSR (rowptr[N+1], col[nb], val[nb]) with every bond listed once
    under its smaller site index.  Draw order: site i ascending, then axis (x first),
    bond (i, i + e_axis mod L)."""
    assert w.model == "ea"
    n, L, D = w.n_sites, w.L, w.dim
    rng = np.random.default_rng(seed)
    nb = n * D
    if w.coupling == "pm1":
        draws = np.where(rng.random(size=nb) < 0.5, 1.0, -1.0).astype(np.float32)
    else:
        draws = rng.normal(0.0, 1.0, size=nb).astype(np.float32)
    coords = site_coords(w)
    strides = np.array([L ** (D - 1 - a) for a in range(D)])
    bonds = {}
    k = 0
    for i in range(n):
        for axis in range(D - 1, -1, -1):          # x (last coordinate) first
            c = coords[i].copy()
            c[axis] = (c[axis] + 1) % L
            j = int((c * strides).sum())
            a, b = (i, j) if i < j else (j, i)
            if a != b:                              # L == 1 degenerate
                bonds[(a, b)] = bonds.get((a, b), np.float32(0.0)) + draws[k]
            k += 1
    keys = sorted(bonds)
    rowptr = np.zeros(n + 1, dtype=np.int32)
    for a, _ in keys:
        rowptr[a + 1] += 1
    rowptr = np.cumsum(rowptr).astype(np.int32)
    col = np.array([b for _, b in keys], dtype=np.int32)
    val = np.array([bonds[kk] for kk in keys], dtype=np.float32)
    return rowptr, col, val


def csr_to_dense_sym(n: int, rowptr, col, val) -> np.ndarray:
    J = np.zeros((n, n), dtype=np.float64)
    for i in range(n):
        for e in range(rowptr[i], rowptr[i + 1]):
            J[i, col[e]] += val[e]
            J[col[e], i] += val[e]
    return J


# ------------------------------------------------------------------------------- masks
def spin_visibility(w: Workload):
    """S_t for every spin t: list of earlier spins it may condition on."""
    n = w.n_sites
    if w.model == "sk" or w.window <= 0:
        return [list(range(t)) for t in range(n)]
    L, D = w.L, w.dim
    strides = [L ** (D - 1 - a) for a in range(D)]
    offs = [o for o in itertools.product(range(-2, 3), repeat=D)
            if 1 <= sum(abs(x) for x in o) <= 2]
    coords = site_coords(w)
    out = []
    for t in range(n):
        s = set(range(max(0, t - w.window), t))
        c = coords[t]
        for o in offs:
            j = sum(((int(c[a]) + o[a]) % L) * strides[a] for a in range(D))
            if j < t:
                s.add(j)
        out.append(sorted(s))
    return out


def make_mask_csr(w: Workload):
    """Position-space CSR (rowptr[N+1], col[nnz]) int32; see module docstring."""
    vis = spin_visibility(w)
    rowptr = np.zeros(w.n_sites + 1, dtype=np.int32)
    cols = []
    for t, s in enumerate(vis):
        row = sorted({j + 1 for j in s if j + 1 <= t} | {t})
        if w.model == "sk" or w.window <= 0:
            row = list(range(t + 1))               # full causal incl. the start position
        cols.extend(row)
        rowptr[t + 1] = len(cols)
    return rowptr, np.asarray(cols, dtype=np.int32)


def band_mask_csr(n: int, width: int):
    """Pure sliding window (Eq. S1): row t = {max(0,t-width) .. t}."""
    rowptr = np.zeros(n + 1, dtype=np.int32)
    cols = []
    for t in range(n):
        cols.extend(range(max(0, t - width), t + 1))
        rowptr[t + 1] = len(cols)
    return rowptr, np.asarray(cols, dtype=np.int32)


def make_all(w: Workload, batch: Optional[int] = None, u_seed: int = SEED_U) -> dict:
    """Everything one run needs, as host numpy arrays."""
    out = {"workload": w, "weights": make_weights(w), "posemb": make_posemb(w),
           "uniforms": make_uniforms(w, batch, u_seed)}
    out["mask_rowptr"], out["mask_col"] = make_mask_csr(w)
    if w.model == "sk":
        out["J"] = make_couplings_sk(w)
    else:
        out["bond_rowptr"], out["bond_col"], out["bond_val"] = make_couplings_ea(spin_lattice(w))
        if w.patch > 1:
            out["site_index"] = patch_site_index(w)
    return out
