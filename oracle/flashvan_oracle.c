/* flashvan_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the FlashVAN hot path computes, written from
 * /root/reference/PAPER.md (arxiv/paper_2606_22984) and the readings listed in DESIGN.md.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_2606_22984_b200/csrc/.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.
 *
 * Pins (tests/test_oracle_pins.py): P1 parameter counts printed in the paper; P2 brute-force
 * sum_s q(s) = 1 for N <= 16; P3 chain rule sample vs log_prob (two separate code paths
 * below); P4 D_KL = beta (F_q - F) >= 0; P5 mask locality; P6 dense == CSR; P7 energy closed
 * forms; P8 zero weights; P9 SK F_inf; P10 head identity; plus an independent restatement
 * with torch CPU library ops (layer_norm, linear, gelu, softmax).  Agreement with the
 * AUTHORS' code (activation, LN eps, LN2 placement) is "parity unpinned": the paper prints
 * no conditional, sample or energy value.
 *
 * Notation follows the paper: N sites, n_l layers, d = d_model, n_h heads, d_h = d / n_h.
 * Positions are 0-based; position t takes the token of spin t-1 (start token 0 at t = 0) and
 * emits the conditional of spin t (Alg. 2).
 *
 * Weights blob (fp32, promoted to fp64 here), row-major [out,in], y = W x + b (Eq. 2, l.98):
 *   tok_emb[V,d_token]; per layer: ln1_g[d] ln1_b[d] Wq[d,d] bq[d] Wk[d,d] bk[d] Wv[d,d] bv[d]
 *   (Wo[d,d] bo[d] iff has_wo) ln2_g[d] ln2_b[d] W1[f,d] b1[f] W2[d,f] b2[d]; head_W[V,d] head_b[V].
 * V = 2 (one spin per token) everywhere except in the patch-token functions at the end of the file, where a
 * token stands for a patch of 2^D spins and V = 2^(2^D) (SI I.D; the parameter counts
 * "w/ patch" of Table 7, l.765-771, fix that the embedding has V rows and the head V logits and biases).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t n_sites, n_layers, d_model, n_heads, d_token, ffn_mult, has_wo, act, ln2_style;
    double ln_eps;
    int32_t vocab;      /* tokens: 2 for one spin per token; 2^(2^D) with 2^D-spin patches (l.603-605) */
} fvo_config;

typedef struct {
    const float *ln1_g, *ln1_b, *wq, *bq, *wk, *bk, *wv, *bv, *wo, *bo, *ln2_g, *ln2_b,
        *w1, *b1, *w2, *b2;
} layer_w;

typedef struct {
    const float *tok_emb;
    layer_w *layer;
    const float *head_w, *head_b;
} model_w;

static int64_t blob_size(const fvo_config *c) {
    int64_t d = c->d_model, f = (int64_t)c->ffn_mult * d;
    int64_t per = 2 * d + 3 * (d * d + d) + (c->has_wo ? d * d + d : 0) + 2 * d + f * d + f + d * f + d;
    return c->vocab * (int64_t)c->d_token + c->n_layers * per + c->vocab * d + c->vocab;
}

int64_t fvo_n_weights(const fvo_config *c) { return blob_size(c); }

static void carve(const fvo_config *c, const float *w, model_w *m) {
    int64_t d = c->d_model, f = (int64_t)c->ffn_mult * d;
    m->tok_emb = w; w += c->vocab * c->d_token;
    for (int l = 0; l < c->n_layers; ++l) {
        layer_w *L = &m->layer[l];
        L->ln1_g = w; w += d; L->ln1_b = w; w += d;
        L->wq = w; w += d * d; L->bq = w; w += d;
        L->wk = w; w += d * d; L->bk = w; w += d;
        L->wv = w; w += d * d; L->bv = w; w += d;
        if (c->has_wo) { L->wo = w; w += d * d; L->bo = w; w += d; } else { L->wo = 0; L->bo = 0; }
        L->ln2_g = w; w += d; L->ln2_b = w; w += d;
        L->w1 = w; w += f * d; L->b1 = w; w += f;
        L->w2 = w; w += d * f; L->b2 = w; w += d;
    }
    m->head_w = w; w += c->vocab * d; m->head_b = w;
}

/* LayerNorm over the feature axis: mean, BIASED variance, eps inside the sqrt, affine.
 * (PAPER.md:235, 339 name the op only; details are reading A6.) */
static void layer_norm(int d, const double *x, const float *g, const float *b, double eps, double *y) {
    double mean = 0.0, var = 0.0;
    for (int i = 0; i < d; ++i) mean += x[i];
    mean /= d;
    for (int i = 0; i < d; ++i) var += (x[i] - mean) * (x[i] - mean);
    var /= d;
    double rstd = 1.0 / sqrt(var + eps);
    for (int i = 0; i < d; ++i) y[i] = (x[i] - mean) * rstd * (double)g[i] + (double)b[i];
}

/* y = W x + b, W row-major [out,in] (Eq. 2). */
static void linear(int out, int in, const float *W, const float *b, const double *x, double *y) {
    for (int o = 0; o < out; ++o) {
        double acc = (double)b[o];
        const float *row = W + (int64_t)o * in;
        for (int i = 0; i < in; ++i) acc += (double)row[i] * x[i];
        y[o] = acc;
    }
}

/* exact GELU 0.5 x (1 + erf(x / sqrt 2))  (reading A5: the paper says "FFN" only). */
static double gelu(double x) { return 0.5 * x * (1.0 + erf(x * 0.70710678118654752440)); }

/* Concatenated positional embedding x = [Embed(token); Embed(position)] (Eq. 15, l.287-292). */
static void embed(const fvo_config *c, const model_w *m, const float *posemb, int tok, int t, double *x) {
    int dt = c->d_token, dp = c->d_model - c->d_token;
    for (int i = 0; i < dt; ++i) x[i] = (double)m->tok_emb[tok * dt + i];
    for (int i = 0; i < dp; ++i) x[dt + i] = (double)posemb[(int64_t)t * dp + i];
}

/* One query against the listed key positions: per head, softmax_j(q.k_j / sqrt(d_h)) v_j,
 * heads concatenated (Eq. 3, l.102-105).  K, V are [N, d] for one sample and layer. */
static void attend(const fvo_config *c, const double *q, const double *K, const double *V,
                   const int32_t *cols, int n_cols, double *u, double *score) {
    int d = c->d_model, nh = c->n_heads, dh = d / nh;
    double scale = 1.0 / sqrt((double)dh);
    for (int h = 0; h < nh; ++h) {
        double mx = -INFINITY;
        for (int e = 0; e < n_cols; ++e) {
            const double *k = K + (int64_t)cols[e] * d + h * dh;
            double s = 0.0;
            for (int i = 0; i < dh; ++i) s += q[h * dh + i] * k[i];
            score[e] = s * scale;
            if (score[e] > mx) mx = score[e];
        }
        double den = 0.0;
        for (int e = 0; e < n_cols; ++e) { score[e] = exp(score[e] - mx); den += score[e]; }
        for (int i = 0; i < dh; ++i) u[h * dh + i] = 0.0;
        for (int e = 0; e < n_cols; ++e) {
            const double *v = V + (int64_t)cols[e] * d + h * dh;
            double p = score[e] / den;
            for (int i = 0; i < dh; ++i) u[h * dh + i] += p * v[i];
        }
    }
}

/* h <- h + u (or W_O u + b_O when has_wo; the paper bypasses W_O, l.107), then the FFN block.
 * ln2_style 0 (Alg. 2 l.346): h <- h + FFN(LN2(h)).  ln2_style 1 (Alg. 1 l.237-239):
 * h <- LN2(h); h <- h + FFN(h). */
static void post_attention(const fvo_config *c, const layer_w *L, double *h, const double *u, double *tmp) {
    int d = c->d_model, f = c->ffn_mult * d;
    double *a = tmp, *hid = tmp + d, *out = tmp + d + f;
    if (c->has_wo) { linear(d, d, L->wo, L->bo, u, a); for (int i = 0; i < d; ++i) h[i] += a[i]; }
    else for (int i = 0; i < d; ++i) h[i] += u[i];
    layer_norm(d, h, L->ln2_g, L->ln2_b, c->ln_eps, a);
    if (c->ln2_style == 1) for (int i = 0; i < d; ++i) h[i] = a[i];
    linear(f, d, L->w1, L->b1, a, hid);
    for (int i = 0; i < f; ++i) hid[i] = gelu(hid[i]);
    linear(d, f, L->w2, L->b2, hid, out);
    for (int i = 0; i < d; ++i) h[i] += out[i];
}

/* p(sigma_t = +1) = softmax(z)[1], z = W_head h + b_head in R^2 (l.243-245, 355-358). */
static double head_p_up(const fvo_config *c, const model_w *m, const double *h) {
    double z[2];
    linear(2, c->d_model, m->head_w, m->head_b, h, z);
    double mx = z[0] > z[1] ? z[0] : z[1];
    double e0 = exp(z[0] - mx), e1 = exp(z[1] - mx);
    return e1 / (e0 + e1);
}

/* log softmax(z)[0], [1]  (Alg. 1 l.9: log q = sum_i log softmax(z_i)[sigma_i]). */
static void head_logp(const fvo_config *c, const model_w *m, const double *h, double *lp_dn, double *lp_up) {
    double z[2];
    linear(2, c->d_model, m->head_w, m->head_b, h, z);
    double mx = z[0] > z[1] ? z[0] : z[1];
    double lse = mx + log(exp(z[0] - mx) + exp(z[1] - mx));
    *lp_dn = z[0] - lse;
    *lp_up = z[1] - lse;
}

/* ---------------------------------------------------------------------------------------
 * Alg. 2: KV-cached ancestral sampling, one site at a time.
 * s_t = +1 iff u_t < p_t(+1) (reading A10); log q accumulates log p_t(s_t).
 * k_t, v_t are appended BEFORE the attention of position t so that t attends itself
 * (Eq. 3 sums j = 1..t; reading A2).
 * spins [B,N] int8 out, logq [B] out, cond_p [B,N] out (may be NULL).
 * ------------------------------------------------------------------------------------- */
int fvo_sample(const fvo_config *c, const float *weights, const float *posemb,
               const int32_t *rowptr, const int32_t *col, int32_t B, const float *uniforms,
               int8_t *spins, double *logq, double *cond_p) {
    int N = c->n_sites, d = c->d_model, f = c->ffn_mult * d, nl = c->n_layers;
    int err = 0;
#pragma omp parallel
    {
        layer_w *lw = (layer_w *)malloc(sizeof(layer_w) * nl);
        model_w m; m.layer = lw; carve(c, weights, &m);
        double *K = (double *)malloc(sizeof(double) * (size_t)nl * N * d);
        double *V = (double *)malloc(sizeof(double) * (size_t)nl * N * d);
        double *h = (double *)malloc(sizeof(double) * (5 * d + 2 * f + N));
        double *a = h + d, *q = a + d, *u = q + d, *tmp = u + d, *score = tmp + 2 * d + f;
        if (!K || !V || !h) {
#pragma omp atomic write
            err = -1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int b = 0; b < B; ++b) {
                double lq = 0.0;
                int prev_tok = 0;                                   /* start token, l.323 */
                for (int t = 0; t < N; ++t) {
                    embed(c, &m, posemb, prev_tok, t, h);           /* l.335 */
                    for (int l = 0; l < nl; ++l) {
                        const layer_w *L = &lw[l];
                        double *Kl = K + (size_t)l * N * d, *Vl = V + (size_t)l * N * d;
                        layer_norm(d, h, L->ln1_g, L->ln1_b, c->ln_eps, a);     /* l.339 */
                        linear(d, d, L->wq, L->bq, a, q);                        /* l.340 */
                        linear(d, d, L->wk, L->bk, a, Kl + (size_t)t * d);
                        linear(d, d, L->wv, L->bv, a, Vl + (size_t)t * d);     /* append, l.349 */
                        attend(c, q, Kl, Vl, col + rowptr[t], rowptr[t + 1] - rowptr[t], u, score);
                        post_attention(c, L, h, u, tmp);                         /* l.344-346 */
                    }
                    double lp_dn, lp_up;
                    head_logp(c, &m, h, &lp_dn, &lp_up);
                    double p_up = head_p_up(c, &m, h);                          /* l.358 */
                    int up = ((double)uniforms[(size_t)b * N + t] < p_up);      /* l.359 */
                    spins[(size_t)b * N + t] = up ? 1 : -1;                     /* l.361 */
                    lq += up ? lp_up : lp_dn;
                    if (cond_p) cond_p[(size_t)b * N + t] = p_up;
                    prev_tok = up;
                }
                logq[b] = lq;
            }
        }
        free(K); free(V); free(h); free(lw);
    }
    return err;
}

/* ---------------------------------------------------------------------------------------
 * Alg. 1: teacher-forced pass, layer by layer over ALL positions.
 * Independent of fvo_sample's loop structure (layer-major here, position-major there),
 * so the chain-rule pin P3 compares two code paths.
 * ------------------------------------------------------------------------------------- */
int fvo_log_prob(const fvo_config *c, const float *weights, const float *posemb,
                 const int32_t *rowptr, const int32_t *col, int32_t B, const int8_t *spins,
                 double *logq, double *cond_p) {
    int N = c->n_sites, d = c->d_model, f = c->ffn_mult * d, nl = c->n_layers;
    int err = 0;
#pragma omp parallel
    {
        layer_w *lw = (layer_w *)malloc(sizeof(layer_w) * nl);
        model_w m; m.layer = lw; carve(c, weights, &m);
        double *X = (double *)malloc(sizeof(double) * (size_t)N * d * 4);
        double *Q = X + (size_t)N * d, *K = Q + (size_t)N * d, *V = K + (size_t)N * d;
        double *a = (double *)malloc(sizeof(double) * (4 * d + 2 * f + N));
        double *u = a + d, *tmp = u + d, *score = tmp + 2 * d + f;
        if (!X || !a) {
#pragma omp atomic write
            err = -1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int b = 0; b < B; ++b) {
                const int8_t *s = spins + (size_t)b * N;
                for (int t = 0; t < N; ++t)                          /* Alg. 1 l.2 */
                    embed(c, &m, posemb, t == 0 ? 0 : (s[t - 1] + 1) / 2, t, X + (size_t)t * d);
                for (int l = 0; l < nl; ++l) {                       /* Alg. 1 l.3-7 */
                    const layer_w *L = &lw[l];
                    for (int t = 0; t < N; ++t) {
                        layer_norm(d, X + (size_t)t * d, L->ln1_g, L->ln1_b, c->ln_eps, a);
                        linear(d, d, L->wq, L->bq, a, Q + (size_t)t * d);
                        linear(d, d, L->wk, L->bk, a, K + (size_t)t * d);
                        linear(d, d, L->wv, L->bv, a, V + (size_t)t * d);
                    }
                    for (int t = 0; t < N; ++t) {
                        attend(c, Q + (size_t)t * d, K, V, col + rowptr[t], rowptr[t + 1] - rowptr[t], u, score);
                        post_attention(c, L, X + (size_t)t * d, u, tmp);
                    }
                }
                double lq = 0.0;
                for (int t = 0; t < N; ++t) {                        /* Alg. 1 l.8-9 */
                    double lp_dn, lp_up;
                    head_logp(c, &m, X + (size_t)t * d, &lp_dn, &lp_up);
                    lq += s[t] > 0 ? lp_up : lp_dn;
                    if (cond_p) cond_p[(size_t)b * N + t] = head_p_up(c, &m, X + (size_t)t * d);
                }
                logq[b] = lq;
            }
        }
        free(X); free(a); free(lw);
    }
    return err;
}

/* E = - sum_{i<j} J_ij s_i s_j by the explicit double loop (Eq. 6; the
 * 1/sqrt(N) of Eq. 6 is folded into J, reading A15). */
void fvo_energy_dense(int32_t B, int32_t N, const int8_t *spins, const float *J, double *E) {
#pragma omp parallel for schedule(static)
    for (int b = 0; b < B; ++b) {
        const int8_t *s = spins + (size_t)b * N;
        double e = 0.0;
        for (int i = 0; i < N; ++i)
            for (int j = i + 1; j < N; ++j) e -= (double)J[(size_t)i * N + j] * s[i] * s[j];
        E[b] = e;
    }
}

/* E = - sum_{<ij>} J_ij s_i s_j, loop over the bond list, each bond once (Eq. 8, l.168). */
void fvo_energy_csr(int32_t B, int32_t N, const int8_t *spins, const int32_t *rowptr,
                    const int32_t *col, const float *val, double *E) {
#pragma omp parallel for schedule(static)
    for (int b = 0; b < B; ++b) {
        const int8_t *s = spins + (size_t)b * N;
        double e = 0.0;
        for (int i = 0; i < N; ++i)
            for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) e -= (double)val[k] * s[i] * s[col[k]];
        E[b] = e;
    }
}

/* =======================================================================================
 * Patch tokens (SI I.D): "the input spin configuration on an L^D lattice is
 * partitioned into non-overlapping patches of size 2^D.  Each patch is mapped to a token, reducing
 * the input sequence length from L^D to (L/2)^D."  The model is unchanged except for its two ends:
 * the embedding table has V = 2^(2^D) rows and the head emits V logits (parameter counts of Table 7,
 * l.765-771).  A token is drawn from Categorical(softmax(z)) (Alg. 2 l.358-359); with a caller-supplied
 * uniform that is the inverse-CDF rule in token order: the first k with u < p_0 + ... + p_k (reading
 * A10 carried over; the last token if rounding leaves u above the total).  Which bit of a token is
 * which spin of the patch is an index list of the workload (workloads.py), not part of this file.
 * probs [B,N,V] (may be NULL) receives the full conditional distribution of every position.
 * ===================================================================================== */
static void head_probs(const fvo_config *c, const model_w *m, const double *h, double *z) {
    int V = c->vocab;
    linear(V, c->d_model, m->head_w, m->head_b, h, z);
    double mx = z[0];
    for (int k = 1; k < V; ++k) if (z[k] > mx) mx = z[k];
    double den = 0.0;
    for (int k = 0; k < V; ++k) { z[k] = exp(z[k] - mx); den += z[k]; }
    for (int k = 0; k < V; ++k) z[k] /= den;
}

int fvo_tok_sample(const fvo_config *c, const float *weights, const float *posemb,
                   const int32_t *rowptr, const int32_t *col, int32_t B, const float *uniforms,
                   int32_t *tokens, double *logq, double *probs) {
    int N = c->n_sites, d = c->d_model, f = c->ffn_mult * d, nl = c->n_layers, V = c->vocab;
    int err = 0;
#pragma omp parallel
    {
        layer_w *lw = (layer_w *)malloc(sizeof(layer_w) * nl);
        model_w m; m.layer = lw; carve(c, weights, &m);
        double *K = (double *)malloc(sizeof(double) * (size_t)nl * N * d);
        double *Vv = (double *)malloc(sizeof(double) * (size_t)nl * N * d);
        double *h = (double *)malloc(sizeof(double) * (5 * d + 2 * f + N + V));
        double *a = h + d, *q = a + d, *u = q + d, *tmp = u + d, *score = tmp + 2 * d + f, *p = score + N;
        if (!K || !Vv || !h) {
#pragma omp atomic write
            err = -1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int b = 0; b < B; ++b) {
                double lq = 0.0;
                int prev_tok = 0;                                   /* start token, l.323 */
                for (int t = 0; t < N; ++t) {
                    embed(c, &m, posemb, prev_tok, t, h);
                    for (int l = 0; l < nl; ++l) {
                        const layer_w *L = &lw[l];
                        double *Kl = K + (size_t)l * N * d, *Vl = Vv + (size_t)l * N * d;
                        layer_norm(d, h, L->ln1_g, L->ln1_b, c->ln_eps, a);
                        linear(d, d, L->wq, L->bq, a, q);
                        linear(d, d, L->wk, L->bk, a, Kl + (size_t)t * d);
                        linear(d, d, L->wv, L->bv, a, Vl + (size_t)t * d);
                        attend(c, q, Kl, Vl, col + rowptr[t], rowptr[t + 1] - rowptr[t], u, score);
                        post_attention(c, L, h, u, tmp);
                    }
                    head_probs(c, &m, h, p);                                   /* l.358 */
                    double uu = (double)uniforms[(size_t)b * N + t], cdf = 0.0;
                    int tok = V - 1;
                    for (int k = 0; k < V; ++k) { cdf += p[k]; if (uu < cdf) { tok = k; break; } }   /* l.359 */
                    tokens[(size_t)b * N + t] = tok;
                    lq += log(p[tok]);
                    if (probs) for (int k = 0; k < V; ++k) probs[((size_t)b * N + t) * V + k] = p[k];
                    prev_tok = tok;
                }
                logq[b] = lq;
            }
        }
        free(K); free(Vv); free(h); free(lw);
    }
    return err;
}

int fvo_tok_log_prob(const fvo_config *c, const float *weights, const float *posemb,
                     const int32_t *rowptr, const int32_t *col, int32_t B, const int32_t *tokens,
                     double *logq, double *probs) {
    int N = c->n_sites, d = c->d_model, f = c->ffn_mult * d, nl = c->n_layers, V = c->vocab;
    int err = 0;
#pragma omp parallel
    {
        layer_w *lw = (layer_w *)malloc(sizeof(layer_w) * nl);
        model_w m; m.layer = lw; carve(c, weights, &m);
        double *X = (double *)malloc(sizeof(double) * (size_t)N * d * 4);
        double *Q = X + (size_t)N * d, *K = Q + (size_t)N * d, *Vv = K + (size_t)N * d;
        double *a = (double *)malloc(sizeof(double) * (4 * d + 2 * f + N + V));
        double *u = a + d, *tmp = u + d, *score = tmp + 2 * d + f, *p = score + N;
        if (!X || !a) {
#pragma omp atomic write
            err = -1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int b = 0; b < B; ++b) {
                const int32_t *s = tokens + (size_t)b * N;
                for (int t = 0; t < N; ++t) embed(c, &m, posemb, t == 0 ? 0 : s[t - 1], t, X + (size_t)t * d);
                for (int l = 0; l < nl; ++l) {
                    const layer_w *L = &lw[l];
                    for (int t = 0; t < N; ++t) {
                        layer_norm(d, X + (size_t)t * d, L->ln1_g, L->ln1_b, c->ln_eps, a);
                        linear(d, d, L->wq, L->bq, a, Q + (size_t)t * d);
                        linear(d, d, L->wk, L->bk, a, K + (size_t)t * d);
                        linear(d, d, L->wv, L->bv, a, Vv + (size_t)t * d);
                    }
                    for (int t = 0; t < N; ++t) {
                        attend(c, Q + (size_t)t * d, K, Vv, col + rowptr[t], rowptr[t + 1] - rowptr[t], u, score);
                        post_attention(c, L, X + (size_t)t * d, u, tmp);
                    }
                }
                double lq = 0.0;
                for (int t = 0; t < N; ++t) {
                    head_probs(c, &m, X + (size_t)t * d, p);
                    lq += log(p[s[t]]);
                    if (probs) for (int k = 0; k < V; ++k) probs[((size_t)b * N + t) * V + k] = p[k];
                }
                logq[b] = lq;
            }
        }
        free(X); free(a); free(lw);
    }
    return err;
}
