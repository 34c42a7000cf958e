"""Thin ctypes binding over libflashvan.so (include/flashvan.h) -- argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels; torch is used for device
memory and streams.  There is no CPU fallback: if the library is missing or the device is not
a B200-class GPU the calls raise.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("FLASHVAN_LIB") or os.path.join(_HERE, "libflashvan.so")

SYMBOLS = ["fv_create_model", "fv_sample", "fv_log_prob", "fv_log_prob_static", "fv_energy_csr", "fv_energy_dense",
           "fv_free_energy", "fv_destroy_model", "fv_n_weights", "fv_kv_bytes", "fv_kv_window", "fv_launch_count",
           "fv_last_error", "fv_markov_mask", "fv_overlap", "fv_lmc_sweeps", "fv_profile", "fv_sampler_kind", "fv_tokens_to_spins"]


class FvConfig(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in
                ("n_sites", "n_layers", "d_model", "n_heads", "d_token", "ffn_mult", "has_wo", "act",
                 "ln2_style", "max_batch", "vocab")] + [("ln_eps", ctypes.c_float)]


class FlashVanError(RuntimeError):
    pass


_lib = None


def lib() -> ctypes.CDLL:
    """Load libflashvan.so (built in-tree by build.py / __graft_entry__.build()); fail loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise FlashVanError(f"{_LIB_PATH} is missing: run `python -m paper_2606_22984_b200.build` "
                                "(there is no CPU fallback)")
        L = ctypes.CDLL(_LIB_PATH)
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
        L.fv_create_model.argtypes = [ctypes.POINTER(FvConfig), vp, i64, vp, vp, vp, vp, ctypes.POINTER(vp)]
        L.fv_sample.argtypes = [vp, i32, vp, vp, vp, vp, vp]
        L.fv_log_prob.argtypes = [vp, i32, vp, vp, vp, vp]
        L.fv_log_prob_static.argtypes = [vp, i32, vp, vp, vp, vp]
        L.fv_energy_csr.argtypes = [i32, i32, vp, vp, vp, vp, i32, vp, vp]
        L.fv_energy_dense.argtypes = [i32, i32, vp, vp, vp, vp]
        L.fv_free_energy.argtypes = [i32, vp, vp, ctypes.c_double, vp, vp]
        L.fv_destroy_model.argtypes = [vp]
        L.fv_destroy_model.restype = None
        L.fv_n_weights.argtypes = [ctypes.POINTER(FvConfig)]
        L.fv_n_weights.restype = i64
        L.fv_kv_bytes.argtypes = [vp]
        L.fv_kv_bytes.restype = i64
        L.fv_kv_window.argtypes = [vp]
        L.fv_kv_window.restype = ctypes.c_int32
        L.fv_launch_count.restype = i64
        L.fv_last_error.restype = ctypes.c_char_p
        L.fv_lmc_sweeps.argtypes = [i32, i32, i32, vp, vp, vp, vp, ctypes.c_float, vp, vp, vp]
        L.fv_overlap.argtypes = [i32, i32, vp, vp, vp, vp, vp]
        L.fv_profile.argtypes = [i32, vp, vp]
        L.fv_tokens_to_spins.argtypes = [i32, i32, i32, vp, vp, vp, vp]
        L.fv_sampler_kind.argtypes = [vp, i32]
        L.fv_sampler_kind.restype = ctypes.c_char_p
        L.fv_markov_mask.argtypes = [i32, i64, vp, vp, i32, vp, vp, i64, ctypes.POINTER(i64), ctypes.POINTER(i32)]
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise FlashVanError(f"{what} failed ({rc}): {lib().fv_last_error().decode()}")


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _dev(t: torch.Tensor, dtype) -> torch.Tensor:
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise FlashVanError(f"expected a contiguous CUDA tensor of {dtype}, got {t.dtype} on {t.device}")
    return t


def _out(t: torch.Tensor, dtype, shape, like: torch.Tensor) -> torch.Tensor:
    """A caller-supplied output buffer: same checks as the inputs, plus shape and device."""
    _dev(t, dtype)
    if tuple(t.shape) != tuple(shape) or t.device != like.device:
        raise FlashVanError(f"output buffer must be {tuple(shape)} on {like.device}, got {tuple(t.shape)} on {t.device}")
    return t


def launch_count() -> int:
    return int(lib().fv_launch_count())


PROFILE_KINDS = ("sample", "lp_qkv", "lp_attn", "lp_ffn", "lp_head")


def profile(enable: bool) -> dict:
    """fv_profile: {kind: (ms, launches)} accumulated since the last call; then switch the timing on or off."""
    ms, n = (ctypes.c_double * 5)(), (ctypes.c_int64 * 5)()
    _check(lib().fv_profile(1 if enable else 0, ms, n), "fv_profile")
    return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(PROFILE_KINDS)}


def make_config(w, max_batch: int) -> FvConfig:
    """`w` is any object with the Workload fields (n_sites, n_layers, d_model, ...)."""
    return FvConfig(w.n_sites, w.n_layers, w.d_model, w.n_heads, w.d_token, w.ffn_mult, w.has_wo, 0,
                    w.ln2_style, max_batch, int(getattr(w, "vocab", 2)), float(w.ln_eps))


class Model:
    """Owner of an `fv_model*`.  create_model / sample / log_prob mirror the C entry points."""

    def __init__(self, cfg: FvConfig, weights, mask_rowptr, mask_col, posemb):
        weights = np.ascontiguousarray(weights, np.float32)
        rp = np.ascontiguousarray(mask_rowptr, np.int32)
        col = np.ascontiguousarray(mask_col, np.int32)
        pe = np.ascontiguousarray(posemb, np.float32)
        if rp.size != cfg.n_sites + 1 or pe.size != cfg.n_sites * (cfg.d_model - cfg.d_token):
            raise FlashVanError("mask_rowptr / posemb size does not match the configuration")
        if col.size != int(rp[-1]):
            raise FlashVanError("mask_col size != mask_rowptr[N]")
        self.cfg = cfg
        self._h = ctypes.c_void_p()
        torch.cuda.init()
        self.device = torch.device("cuda", torch.cuda.current_device())   # the KV pool lives here
        _check(lib().fv_create_model(ctypes.byref(cfg), weights.ctypes.data, weights.size, rp.ctypes.data,
                                     col.ctypes.data, pe.ctypes.data, _stream(), ctypes.byref(self._h)),
               "fv_create_model")

    @property
    def kv_bytes(self) -> int:
        return int(lib().fv_kv_bytes(self._h))

    @property
    def kv_window(self) -> int:
        """Rows of fv_sample's ring-buffer KV window for a band mask (Eq. S1), 0 for any other mask."""
        return int(lib().fv_kv_window(self._h))

    def sample(self, uniforms: torch.Tensor, want_cond_p: bool = False, out=None):
        """fv_sample: uniforms [B,N] f32 cuda -> (spins int8 [B,N], logq f32 [B], cond_p or None)."""
        u = _dev(uniforms, torch.float32)
        B, N = u.shape
        if N != self.cfg.n_sites or u.device != self.device:
            raise FlashVanError(f"uniforms must be [B, n_sites] on {self.device}")
        if out is None:
            spins = torch.empty((B, N), dtype=torch.int8, device=u.device)
            logq = torch.empty((B,), dtype=torch.float32, device=u.device)
        else:
            spins, logq = _out(out[0], torch.int8, (B, N), u), _out(out[1], torch.float32, (B,), u)
        cp = torch.empty((B, N), dtype=torch.float32, device=u.device) if want_cond_p else None
        _check(lib().fv_sample(self._h, B, u.data_ptr(), spins.data_ptr(), logq.data_ptr(),
                               cp.data_ptr() if cp is not None else None, _stream()), "fv_sample")
        return spins, logq, cp

    def log_prob(self, spins: torch.Tensor, want_cond_p: bool = False, out=None):
        """fv_log_prob: spins int8 [B,N] cuda -> (logq f32 [B], cond_p or None)."""
        s = _dev(spins, torch.int8)
        B, N = s.shape
        if N != self.cfg.n_sites or s.device != self.device:
            raise FlashVanError(f"spins must be [B, n_sites] on {self.device}")
        logq = torch.empty((B,), dtype=torch.float32, device=s.device) if out is None else _out(out, torch.float32, (B,), s)
        cp = torch.empty((B, N), dtype=torch.float32, device=s.device) if want_cond_p else None
        _check(lib().fv_log_prob(self._h, B, s.data_ptr(), logq.data_ptr(),
                                 cp.data_ptr() if cp is not None else None, _stream()), "fv_log_prob")
        return logq, cp

    def log_prob_static(self, spins: torch.Tensor, logq: torch.Tensor, cond_p: torch.Tensor = None):
        """fv_log_prob_static: fv_log_prob with its workspace in the library's static device array -- no allocation,
        here or in the library (the caller passes the outputs: logq f32 [B], cond_p f32 [B,N] or None).  Calls that
        overlap on the GPU race on that array; B * N is limited (flashvan.h: FV_STATIC_SCRATCH_BYTES)."""
        s = _dev(spins, torch.int8)
        B, N = s.shape
        if N != self.cfg.n_sites or s.device != self.device:
            raise FlashVanError(f"spins must be [B, n_sites] on {self.device}")
        logq = _out(logq, torch.float32, (B,), s)
        cp = _out(cond_p, torch.float32, (B, N), s) if cond_p is not None else None
        _check(lib().fv_log_prob_static(self._h, B, s.data_ptr(), logq.data_ptr(),
                                        cp.data_ptr() if cp is not None else None, _stream()), "fv_log_prob_static")
        return logq, cp

    def sampler_kind(self, B: int) -> str:
        """Which of the two fv_sample kernels a batch of B takes: "chain" or "ring"."""
        return lib().fv_sampler_kind(self._h, B).decode()

    def close(self):
        if self._h:
            lib().fv_destroy_model(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def create_model(w, weights, mask_rowptr, mask_col, posemb, max_batch: int) -> Model:
    return Model(make_config(w, max_batch), weights, mask_rowptr, mask_col, posemb)


def energy_csr(spins, rowptr, col, val, integer_couplings: bool, out=None):
    s = _dev(spins, torch.int8)
    B, N = s.shape
    E = torch.empty((B,), dtype=torch.float32, device=s.device) if out is None else _out(out, torch.float32, (B,), s)
    _check(lib().fv_energy_csr(B, N, s.data_ptr(), _dev(rowptr, torch.int32).data_ptr(),
                               _dev(col, torch.int32).data_ptr(), _dev(val, torch.float32).data_ptr(),
                               1 if integer_couplings else 0, E.data_ptr(), _stream()), "fv_energy_csr")
    return E


def energy_dense(spins, J, out=None):
    s = _dev(spins, torch.int8)
    B, N = s.shape
    J = _dev(J, torch.float32)
    if tuple(J.shape) != (N, N):
        raise FlashVanError("J must be [N, N]")
    E = torch.empty((B,), dtype=torch.float32, device=s.device) if out is None else _out(out, torch.float32, (B,), s)
    _check(lib().fv_energy_dense(B, N, s.data_ptr(), J.data_ptr(), E.data_ptr(), _stream()), "fv_energy_dense")
    return E


def free_energy(E, logq, temperature: float, out=None):
    """fv_free_energy: returns a 4-element f64 CUDA tensor (mean, population std of L = E + T log q, count,
    sum of squared deviations)."""
    E, logq = _dev(E, torch.float32), _dev(logq, torch.float32)
    if E.shape != logq.shape or E.dim() != 1:
        raise FlashVanError("free_energy: E and logq must be [B]")
    res = torch.empty((4,), dtype=torch.float64, device=E.device) if out is None else _out(out, torch.float64, (4,), E)
    _check(lib().fv_free_energy(E.numel(), E.data_ptr(), logq.data_ptr(), float(temperature),
                                res.data_ptr(), _stream()), "fv_free_energy")
    return res


def lmc_sweeps(spins, adj_rowptr, adj_col, adj_val, beta: float, exp_variates):
    """fv_lmc_sweeps: Metropolis sweeps in place on `spins` (int8 CUDA tensor [B, N]); exp_variates fp32
    [B, n_sweeps, N].  Returns the accepted-flip counts (int32 [B])."""
    if spins.dtype != torch.int8 or not spins.is_cuda or not spins.is_contiguous() or spins.dim() != 2:
        raise FlashVanError("lmc_sweeps: spins must be a contiguous int8 CUDA tensor [B, N] (updated in place)")
    B, N = spins.shape
    ev = _dev(exp_variates, torch.float32)
    if ev.dim() != 3 or ev.shape[0] != B or ev.shape[2] != N:
        raise FlashVanError("lmc_sweeps: exp_variates must be [B, n_sweeps, N]")
    rp, col, val = _dev(adj_rowptr, torch.int32), _dev(adj_col, torch.int32), _dev(adj_val, torch.float32)
    acc = torch.empty((B,), dtype=torch.int32, device=spins.device)
    _check(lib().fv_lmc_sweeps(B, N, ev.shape[1], spins.data_ptr(), rp.data_ptr(), col.data_ptr(), val.data_ptr(),
                               float(beta), ev.data_ptr(), acc.data_ptr(), _stream()), "fv_lmc_sweeps")
    return acc


def tokens_to_spins(tokens, site_index):
    """fv_tokens_to_spins: patch tokens (uint8 or int8 storage, [B, n_tokens] CUDA) -> lattice spins int8
    [B, n_tokens * P]; site_index int32 [n_tokens, P] CUDA (bit k of token n is the spin of that lattice site)."""
    if tokens.dtype not in (torch.uint8, torch.int8) or not tokens.is_cuda or not tokens.is_contiguous() or tokens.dim() != 2:
        raise FlashVanError("tokens_to_spins: tokens must be a contiguous byte CUDA tensor [B, n_tokens]")
    si = _dev(site_index, torch.int32)
    B, n_tok = tokens.shape
    if si.dim() != 2 or si.shape[0] != n_tok or not 1 <= si.shape[1] <= 8:
        raise FlashVanError("tokens_to_spins: site_index must be [n_tokens, P] with P <= 8")
    P = si.shape[1]
    spins = torch.empty((B, n_tok * P), dtype=torch.int8, device=tokens.device)
    _check(lib().fv_tokens_to_spins(B, n_tok, P, tokens.data_ptr(), si.data_ptr(), spins.data_ptr(), _stream()),
           "fv_tokens_to_spins")
    return spins


def overlap(spins_a, spins_b, want_hist: bool = True):
    """fv_overlap: (dot int32 [B], hist int32 [N + 1] or None); q = dot / N (Eq. 9)."""
    a, c = _dev(spins_a, torch.int8), _dev(spins_b, torch.int8)
    if a.shape != c.shape or a.dim() != 2:
        raise FlashVanError("overlap: two [B, N] int8 tensors of one shape")
    B, N = a.shape
    dot = torch.empty((B,), dtype=torch.int32, device=a.device)
    hist = torch.empty((N + 1,), dtype=torch.int32, device=a.device) if want_hist else None
    _check(lib().fv_overlap(B, N, a.data_ptr(), c.data_ptr(), dot.data_ptr(),
                            hist.data_ptr() if want_hist else None, _stream()), "fv_overlap")
    return dot, hist


def markov_mask(n: int, edge_a, edge_b, position_space: bool = True):
    """Ordered Markov boundary of every vertex as CSR (host numpy in, host numpy out): the mask
    create_model takes when position_space, else the boundary sets themselves.  Returns
    (rowptr int32 [n+1], col int32 [nnz], d_max)."""
    import numpy as np
    a = np.ascontiguousarray(edge_a, dtype=np.int32)
    b = np.ascontiguousarray(edge_b, dtype=np.int32)
    if a.shape != b.shape or a.ndim != 1:
        raise FlashVanError("markov_mask: edge_a and edge_b must be 1-D arrays of one length")
    rowptr = np.zeros(n + 1, dtype=np.int32)
    nnz, dmax = ctypes.c_int64(0), ctypes.c_int32(0)
    args = (n, a.size, a.ctypes.data if a.size else None, b.ctypes.data if b.size else None, int(bool(position_space)))
    rc = lib().fv_markov_mask(*args, rowptr.ctypes.data, None, 0, ctypes.byref(nnz), ctypes.byref(dmax))
    if rc != 0 and nnz.value == 0:
        _check(rc, "fv_markov_mask")
    col = np.zeros(max(nnz.value, 1), dtype=np.int32)
    _check(lib().fv_markov_mask(*args, rowptr.ctypes.data, col.ctypes.data, nnz.value, ctypes.byref(nnz),
                                ctypes.byref(dmax)), "fv_markov_mask")
    return rowptr, col[:nnz.value], dmax.value
