/* flashvan.h -- C-ABI of libflashvan.so: the B200 (sm_100a) hot path of FlashVAN
 * (arxiv/paper_2606_22984): KV-cached ancestral sampling under a per-site CSR attention
 * mask, the teacher-forced log q(s) pass, and the batched Ising energy.
 *
 * Citations are PAPER.md line + the section / equation / algorithm the line falls in.
 * Readings of silent or garbled passages are numbered A1..A21 in DESIGN.md.
 *
 * General rules
 *   - Every array argument marked [device] is a CUDA device pointer allocated by the caller
 *     and borrowed for the call; arguments marked [host] are host pointers.  The library
 *     never frees caller memory.  fv_create_model copies what it keeps.
 *   - `stream` is a cudaStream_t passed as void*.  fv_sample, fv_log_prob, fv_energy_* and
 *     fv_free_energy only enqueue work on it and never synchronise the device;
 *     fv_create_model / fv_destroy_model synchronise.
 *   - Return value: 0 on success, a negative FV_ERR_* otherwise; fv_last_error() then gives a
 *     thread-local message.  Outputs are unspecified after an error.  There is no CPU
 *     fallback and no other backend: a non-sm_100 device is FV_ERR_ARCH.
 *   - Results are bit-reproducible run to run for fixed inputs (no float atomics).
 *   - 0-based positions.  Position t takes the token of spin t-1 (start token 0 for t = 0,
 *     sharing id 0 with spin -1) and emits the conditional of spin t (PAPER.md:314-363,
 *     Alg. 2 l.6-11; reading A3).
 */
#ifndef FLASHVAN_H
#define FLASHVAN_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FV_OK 0
#define FV_ERR_BAD_ARG (-1)   /* NULL pointer, non-positive size, B > max_batch            */
#define FV_ERR_BAD_MASK (-2)  /* row not ascending/unique, col > row, col < 0, last != row  */
#define FV_ERR_BAD_SHAPE (-3) /* unsupported d_model / head size / n_weights mismatch       */
#define FV_ERR_CUDA (-4)      /* a CUDA runtime call failed                                 */
#define FV_ERR_OOM (-5)       /* device allocation failed                                   */
#define FV_ERR_ARCH (-6)      /* current device is not compute capability 10.x              */

typedef struct fv_model fv_model; /* opaque, library-owned */

/* Architecture of the decoder (PAPER.md:92-109 II.A.3; Alg. 1 l.226-246; Alg. 2 l.314-363). */
typedef struct {
    int32_t n_sites;   /* N: sequence length = number of spins                               */
    int32_t n_layers;  /* n_l decoder layers                                                 */
    int32_t d_model;   /* d = d_token + d_pos (Eq. 15 l.287-292); 32, 64, 128 or 256          */
    int32_t n_heads;   /* n_h; d_h = d / n_h must be 8, 16, 32 or 64                          */
    int32_t d_token;   /* token-embedding width (paper default 2, l.577)                     */
    int32_t ffn_mult;  /* FFN hidden width / d; must be 4 (pinned by the paper's counts, P1)  */
    int32_t has_wo;    /* 0: W_O bypassed as in the paper (l.107); 1: u <- W_O u + b_O        */
    int32_t act;       /* 0: exact GELU (reading A5); no other value is defined               */
    int32_t ln2_style; /* 0: h += FFN(LN2(h)) (Alg. 2 l.346); 1: h = LN2(h); h += FFN(h)      */
                       /*    (Alg. 1 l.237-239); reading A1                                   */
    int32_t max_batch; /* KV pool is sized for this many samples                              */
    int32_t vocab;     /* tokens: 2 = one spin per token (0 is read as 2); 16 or 256 = one token  */
                       /*    per patch of 4 / 8 spins (SI I.D, l.603-605; needs d_model <= 128,    */
                       /*    has_wo = 0): embedding and head then have `vocab` rows, tokens are    */
                       /*    drawn by inverse CDF from the one uniform of the position             */
    float ln_eps;      /* LayerNorm epsilon (reading A6: 1e-5)                                */
} fv_config;

/* Build a model object.
 *   weights [host]  n_weights fp32 values in this order, matrices row-major [out,in], y = Wx+b
 *       (Eq. 2, l.98-100): tok_emb[V,d_token] (V = vocab); per layer ln1_g[d] ln1_b[d] Wq[d,d] bq[d]
 *       Wk[d,d] bk[d] Wv[d,d] bv[d] (Wo[d,d] bo[d] iff has_wo) ln2_g[d] ln2_b[d] W1[4d,d]
 *       b1[4d] W2[d,4d] b2[d]; then head_W[V,d] head_b[V].  GEMM operands are rounded to bf16
 *       once here; LayerNorm, biases, embeddings and the head stay fp32.
 *   mask_rowptr [host] N+1, mask_col [host] rowptr[N]: CSR in POSITION space (reading A11):
 *       row t lists the key positions A(t), ascending, unique, all <= t, last entry == t
 *       (Eq. 3 l.102 sums j <= t; Eq. S1 l.555 is the banded special case).
 *   posemb [host] [N, d_model - d_token] fp32 (Eq. 15).
 * Allocates the bf16 KV pool, a dense array [max_batch][n_layers][N] of rows of 2d bf16 (K then V; every
 * sample has the same length, so there is no page table), on the CURRENT device -- every later call that
 * takes the model must be made with that device current (FV_ERR_BAD_ARG otherwise) -- and for
 * d_model <= 128 without W_O the fv_log_prob workspace (two fp32 arrays [max_batch * N, d_model]).
 * Synchronises `stream`.  *out is owned by the library until fv_destroy_model. */
int fv_create_model(const fv_config* cfg, const float* weights, int64_t n_weights,
                    const int32_t* mask_rowptr, const int32_t* mask_col, const float* posemb,
                    void* stream, fv_model** out);

/* Alg. 2: ancestral sampling of B <= max_batch configurations.
 *   uniforms [device] [B,N] fp32 in [0,1): spin t of sample b is +1 iff u[b,t] < p_t(+1)
 *       (strict, compared in fp32; reading A10 replaces Categorical(p_t), l.359).
 *   spins  [device] [B,N] int8 out, values +-1 (l.361: sigma = 2 s - 1).
 *   logq   [device] [B] fp32 out: sum_t log p_t(s_t) (Alg. 1 l.9), accumulated in fp64.
 *   cond_p [device] [B,N] fp32 out or NULL: p_t(+1 | s_<t).
 * With vocab > 2 (patch tokens): `spins` receives the TOKEN of every position as an unsigned byte (0 .. vocab - 1;
 * fv_tokens_to_spins unpacks them onto the lattice), drawn as the first k with u < p_0 + ... + p_k in token
 * order (fp32 softmax over the `vocab` logits; the last token if rounding leaves u above the total); cond_p
 * receives the probability of the drawn token. */
int fv_sample(fv_model* m, int32_t B, const float* uniforms, int8_t* spins, float* logq,
              float* cond_p, void* stream);

/* Alg. 1: teacher-forced log q(s) of given configurations.
 *   spins [device] [B,N] int8 in (+-1; other values are undefined behaviour).
 *   (vocab > 2: token ids as unsigned bytes, cond_p = probability of the given token.)
 *   logq, cond_p as in fv_sample.  Overwrites the model's KV pool and workspace: calls on one model
 *   must be ordered on one stream.  Enqueues 3 * n_layers + 1 kernels (layer-major tensor-core path; 4 * n_layers + 1
 *   with has_wo: the out-projection is one more tcgen05 GEMM per layer) or one (chunked teacher forcing: d_model = 256). */
int fv_log_prob(fv_model* m, int32_t B, const int8_t* spins, float* logq, float* cond_p,
                void* stream);

/* fv_log_prob for callers that must not allocate (CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the same kernels and the same results, bit for bit, but the call's workspace -- the residual stream h
 * and the queries q (fp32 [B*N, d_model] each) and the layer-major K|V rows (bf16 [B][n_layers][N][2 d_model]) -- lives
 * in ONE file-scope `static __device__` array of FV_STATIC_SCRATCH_BYTES inside the library instead of the model's
 * own buffers.  Every GPU that loads the library holds that array until the process exits.  The call itself makes no
 * cudaMalloc / cudaFree / allocating library call (keep fv_profile off: its events are created on demand); the first
 * call on a device looks the array's address up once (cudaGetSymbolAddress).
 *   Limit: B * N * d_model * (8 + 4 * n_layers) bytes (+ alignment) <= FV_STATIC_SCRATCH_BYTES, i.e. 16 384 rows
 *   (B * N) for a 6-layer d_model = 128 model; larger calls return FV_ERR_BAD_ARG and fv_last_error() names the
 *   bytes needed.  Shapes the layer-major path does not cover (d_model = 256) return FV_ERR_BAD_SHAPE.
 *   The array is shared by every model and every call on the device and keeps the previous call's contents; nothing
 *   in it needs clearing (each call writes every row before reading it), but two calls that overlap on the GPU
 *   (different streams, or two host threads) race on it: order them on one stream.  The model's KV pool is untouched.
 * Arguments, outputs and error codes otherwise as fv_log_prob. */
#define FV_STATIC_SCRATCH_BYTES (64u << 20)
int fv_log_prob_static(fv_model* m, int32_t B, const int8_t* spins, float* logq, float* cond_p,
                       void* stream);

/* Eq. 8: E_b = - sum over listed bonds J_ij s_i s_j, every bond listed once.
 *   rowptr [device] N+1, col [device], val [device] fp32: CSR of the bonds (any triangle).
 *   integer_couplings != 0: every val is an integer; the sum is taken in int32 and is exact.
 *   E [device] [B] fp32 out. */
int fv_energy_csr(int32_t B, int32_t N, const int8_t* spins, const int32_t* rowptr,
                  const int32_t* col, const float* val, int32_t integer_couplings, float* E,
                  void* stream);

/* Eq. 6 (1/sqrt(N) folded into J; reading A15): E_b = - sum_{i<j} J_ij s_i s_j
 * = -1/2 s^T J s for symmetric J with zero diagonal.
 *   J [device] [N,N] fp32 row-major, symmetric, zero diagonal.  E [device] [B] fp32 out. */
int fv_energy_dense(int32_t B, int32_t N, const int8_t* spins, const float* J, float* E,
                    void* stream);

/* Eq. 5: L_b = E_b + T logq_b; out[0] = mean_b L_b, out[1] = population std,
 *   out[2] = B, out[3] = sum_b (L_b - mean)^2 (the two a batch-sharded run merges across ranks).
 *   E, logq [device] [B] fp32; out [device] 4 x fp64.  Deterministic single-block fp64 tree. */
int fv_free_energy(int32_t B, const float* E, const float* logq, double temperature, double* out,
                   void* stream);

/* Replica overlap, Eq. 9: q_b = (1/N) sum_i a_bi c_bi between sample b of one set and sample b of
 * another (two independent sampling runs, or the two halves of one).
 *   spins_a, spins_b [device] [B, N] int8 +-1.  dot [device] [B] int32: the exact sum, q_b = dot[b] / N.
 *   hist [device, may be NULL] N + 1 int32 counters, zeroed by the call: hist[(dot + N) / 2] is the number of
 *   samples at each of the values -N, -N + 2, ..., N the sum can take, i.e. p(q) = hist / B.  Integer arithmetic
 *   throughout: bit-exact and order-independent. */
int fv_overlap(int32_t B, int32_t N, const int8_t* spins_a, const int8_t* spins_b, int32_t* dot, int32_t* hist,
               void* stream);

/* Local Monte Carlo refinement of samples (SI I.C l.583-595 "short LMC procedure").  The
 * paper names neither the acceptance rule nor the number of sweeps; this is the textbook Metropolis single-spin
 * flip, n_sweeps sweeps over the sites in index order: h_i = sum_j J_ij s_j in the order the adjacency lists the
 * neighbours (fp32), dE = 2 s_i h_i, flip iff beta * dE < e, e a standard exponential variate (-ln u) supplied
 * by the caller, so P(accept) = min(1, exp(-beta dE)) and the kernel itself draws nothing.
 *   spins [device] [B, N] int8 +-1, updated in place.  adj_rowptr / adj_col / adj_val [device]: FULL symmetric
 *   adjacency CSR (every bond listed at both ends; fv_energy_csr's bond list names each bond once).
 *   exp_variates [device] [B, n_sweeps, N] fp32 >= 0 (may be NULL when n_sweeps = 0).  accepted [device, may be NULL] [B] int32: flips accepted
 *   per sample.  N <= 49152 (a sample's spins stay in shared memory for all sweeps).  Bit-reproducible. */
int fv_lmc_sweeps(int32_t B, int32_t N, int32_t n_sweeps, int8_t* spins, const int32_t* adj_rowptr,
                  const int32_t* adj_col, const float* adj_val, float beta, const float* exp_variates,
                  int32_t* accepted, void* stream);

void fv_destroy_model(fv_model* m);

/* Build the paper's attention mask from the coupling graph: the ordered Markov boundary of every vertex
 * (Sec. IV.A.1, Eq. 12-13), i.e. the past vertices j < i adjacent to i or joined to i
 * by a path through future vertices (> i) only; a sliding window of width W >= d_max contains it
 * (Eq. S1).  Host-only call, no device work.
 *   n: number of vertices, numbered in sampling order.  edge_a, edge_b [host] n_edges undirected edges
 *       (duplicates allowed; a self loop or an index outside [0, n) is FV_ERR_BAD_ARG).
 *   position_space = 0: row i = boundary(i) in vertex indices, ascending (may be empty).
 *   position_space = 1: row t = {j + 1 : j in boundary(t)} U {t}, ascending -- the mask_rowptr / mask_col
 *       fv_create_model takes (position j + 1 carries spin j; reading A11).
 *   out_rowptr [host] n + 1 (always written).  out_col [host] room for `cap` entries; if cap is smaller
 *       than the number of entries needed, nothing is written to out_col and FV_ERR_BAD_ARG is returned
 *       with *nnz set, so a first call with cap = 0 sizes the second.  More than 2^31 - 1 entries is
 *       FV_ERR_BAD_SHAPE.
 *   nnz [host, may be NULL]: entries needed.  d_max [host, may be NULL]: max_i max_{j in boundary(i)} (i - j). */
int fv_markov_mask(int32_t n, int64_t n_edges, const int32_t* edge_a, const int32_t* edge_b,
                   int32_t position_space, int32_t* out_rowptr, int32_t* out_col, int64_t cap,
                   int64_t* nnz, int32_t* d_max);

/* Expected n_weights for a configuration (the layout above); < 0 on a bad shape. */
int64_t fv_n_weights(const fv_config* cfg);

/* Patch tokens -> lattice spins (SI I.D, l.603-605): bit k of token n of sample b is the spin (2 bit - 1, l.361) of
 * lattice site site_index[n * P + k].
 *   tokens [device] [B, n_tokens] unsigned bytes; site_index [device] [n_tokens * P] int32, a permutation of
 *   0 .. n_tokens * P - 1 (P = spins per token <= 8); spins [device] [B, n_tokens * P] int8 out. */
int fv_tokens_to_spins(int32_t B, int32_t n_tokens, int32_t P, const uint8_t* tokens, const int32_t* site_index,
                       int8_t* spins, void* stream);

/* Which fv_sample kernel a batch of B samples takes on this model: "ring-tc" (one CTA per sample group, KV rows and
 * weights streamed through one shared-memory ring, projections on tcgen05: d_model = 128, 16-wide heads, no W_O),
 * "ring" (the same with mma.sync projections: every other shape, or FLASHVAN_DECODE=ring), "chain" (layer-pipelined
 * clusters with the weights resident on chip, FLASHVAN_DECODE=chain); "none" for bad arguments.  A static string. */
const char* fv_sampler_kind(const fv_model* m, int32_t B);

/* Per-kernel device times, for measurement (bench.py's GEMM roofline).  While switched on, the library brackets
 * the launches of each kernel class with CUDA events on the launching stream.  A call returns, and clears, what
 * has accumulated since the previous call, then sets the switch to `enable`:
 *   ms [host, may be NULL] 5 x fp64, launches [host, may be NULL] 5 x int64, in the order
 *   {fv_sample kernel, fv_log_prob: LN1+QKV GEMM, masked attention, fused LN2+FFN GEMMs, head}.
 * Synchronises on the recorded events (i.e. on the work they bracket). */
int fv_profile(int32_t enable, double* ms, int64_t* launches);

/* Bytes of device memory fv_sample's KV pool occupies (0 for NULL). */
int64_t fv_kv_bytes(const fv_model* m);

/* Band-only fast path (Eq. S1: M_ij = 0 iff i - j <= W).  When every mask row t is
 * the single run max(0, t-W)..t and 2(W+1) <= N, fv_create_model gives fv_sample a ring-buffer KV window of W+1 rows per
 * (sample, layer) instead of N rows -- position p lives in row p mod (W+1), results are bit-identical to the N-row pool --
 * and fv_log_prob allocates its own N-row pool at its first call (cudaMalloc: that one call synchronises the device).
 * Returns W+1 for such a model, 0 otherwise (and for NULL).  FLASHVAN_KV=dense in the environment at fv_create_model
 * time keeps the N-row pool (A/B measurements). */
int32_t fv_kv_window(const fv_model* m);

/* Number of kernel launches the library has enqueued since load (for bench.py gpu_launches). */
int64_t fv_launch_count(void);

/* Thread-local message of the last failing call; valid until the next call on the thread. */
const char* fv_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* FLASHVAN_H */
