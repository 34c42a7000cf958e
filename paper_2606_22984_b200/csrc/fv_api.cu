// fv_api.cu -- the extern "C" boundary of libflashvan.so (see include/flashvan.h).
// Host orchestration only: argument validation, one-off weight packing, launch geometry.
#include <algorithm>
#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/flashvan.h"
#include "fv_internal.h"

struct fv_model {
    fv_config cfg;
    FvModelDev dev;
    void* arena = nullptr;       // all read-only parameters, one allocation
    size_t arena_bytes = 0;
    size_t kv_bytes = 0;
    void* ws = nullptr;          // fv_log_prob workspace (h, q)
    size_t ws_bytes = 0;
    int n_sms = 0;
    int device = 0;
    double mean_nnz = 0.0;       // mask entries per row
    int window = 0;              // > 0: band mask, fv_sample's pool is a ring-buffer window of this many rows per stream
    size_t kv_full_bytes = 0;    // fv_log_prob's pool [max_batch][n_layers][N][2d] (window mode: allocated at its first call)
};

namespace {

thread_local std::string g_err;
std::atomic<long long> g_launches{0};

// fv_profile: event pairs per kernel class, filled by fv_prof_begin / fv_prof_end while switched on
std::mutex g_prof_mu;
bool g_prof_on = false;
std::vector<std::pair<cudaEvent_t, cudaEvent_t>> g_prof_ev[FV_K_COUNT];

int fail(int code, const std::string& msg) {
    g_err = msg;
    return code;
}

// Every call that takes an fv_model must run on the device the model (its KV pool, its weights) lives on.
int wrong_device(const fv_model* m) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != m->device)
        return fail(FV_ERR_BAD_ARG, "the model lives on device " + std::to_string(m->device) + ", the current device is " +
                                        std::to_string(dev));
    return 0;
}

// fv_sample's choice between its two kernels, before the shape check of the chain sampler.
bool wants_chain(const fv_model* m) {
    const char* dmode = std::getenv("FLASHVAN_DECODE");
    if (dmode && *dmode) return std::strcmp(dmode, "chain") == 0;
    (void)m;
    return false;             // opt-in until it beats the streaming kernel
}

// The streaming sampler with tcgen05 projections (fv_decode_tc.cu) is the default where it exists (d = 128, 16-wide heads,
// no W_O); FLASHVAN_DECODE=ring keeps the mma.sync kernel of fv_decode.cu for comparison.
// nt = n8-tiles of samples per CTA: with <= 8 samples per CTA the separate MMA / epilogue round trips of the tcgen05 path
// cost more than they save (cfg5: 292 vs 252 ms), from 9 samples per CTA on it wins (cfg4, 28 per CTA: 83.6 vs 91.0 ms).
bool wants_tc(const fv_model* m, int nt) {
    const char* dmode = std::getenv("FLASHVAN_DECODE");
    if (dmode && *dmode) return std::strcmp(dmode, "tc") == 0;
    return nt >= 2 && m->cfg.d_model == 128 && m->cfg.d_model / m->cfg.n_heads == 16 && !m->cfg.has_wo;
}

int cuda_fail(cudaError_t e, const char* what) {
    return fail(e == cudaErrorMemoryAllocation ? FV_ERR_OOM : FV_ERR_CUDA,
                std::string(what) + ": " + cudaGetErrorString(e));
}

bool shape_ok(const fv_config* c) {
    if (!c || c->n_sites <= 0 || c->n_layers <= 0 || c->n_layers > FV_MAX_LAYERS) return false;
    if (c->ffn_mult != 4 || c->act != 0) return false;
    if (c->d_token <= 0 || c->d_token >= c->d_model) return false;
    if (c->n_heads <= 0 || c->d_model % c->n_heads) return false;
    const int dh = c->d_model / c->n_heads;
    const int key = c->d_model * 1000 + dh;
    if (c->vocab != 0 && c->vocab != 2 && !((c->vocab == 16 || c->vocab == 256) && c->d_model <= 128 && !c->has_wo)) return false;
    return key == 32016 || key == 64016 || key == 64032 || key == 128016 || key == 128032 || key == 256064;
}

int64_t n_weights_of(const fv_config* c) {
    const int64_t d = c->d_model, f = 4 * d;
    const int64_t per = 2 * d + 3 * (d * d + d) + (c->has_wo ? d * d + d : 0) + 2 * d + f * d + f + d * f + d;
    const int64_t V = c->vocab > 2 ? c->vocab : 2;
    return V * (int64_t)c->d_token + c->n_layers * per + V * d + V;
}

uint16_t bf16_bits(float x) {
    __nv_bfloat16 h = __float2bfloat16_rn(x);
    uint16_t u;
    std::memcpy(&u, &h, 2);
    return u;
}

// W[out,in] fp32 row-major -> bf16 in mma.m16n8k16 A-fragment order: tile (mt,kt), lane, 8 values
//   reg j/2: a0=(g, 2c..2c+1) a1=(g+8, 2c..) a2=(g, 2c+8..) a3=(g+8, 2c+8..),  g = lane/4, c = lane%4.
void pack_mma_a(const float* W, int out, int in, uint16_t* dst) {
    const int MT = out / 16, KT = in / 16;
    for (int mt = 0; mt < MT; ++mt)
        for (int kt = 0; kt < KT; ++kt)
            for (int lane = 0; lane < 32; ++lane)
                for (int j = 0; j < 8; ++j) {
                    const int reg = j >> 1, half = j & 1, g = lane >> 2, c = lane & 3;
                    const int row = mt * 16 + g + ((reg & 1) ? 8 : 0);
                    const int k = kt * 16 + 2 * c + half + ((reg & 2) ? 8 : 0);
                    dst[(((size_t)mt * KT + kt) * 32 + lane) * 8 + j] = bf16_bits(W[(size_t)row * in + k]);
                }
}

struct Arena {
    std::vector<unsigned char> host;
    size_t reserve(size_t bytes) {
        const size_t off = (host.size() + 255) / 256 * 256;
        host.resize(off + bytes);
        return off;
    }
    size_t put(const void* src, size_t bytes) {
        const size_t off = reserve(bytes);
        std::memcpy(host.data() + off, src, bytes);
        return off;
    }
};

}  // namespace

void fv_prof_begin(int kind, cudaStream_t s) {
    std::lock_guard<std::mutex> lock(g_prof_mu);
    if (!g_prof_on) return;
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
    cudaEventRecord(a, s);
    g_prof_ev[kind].push_back({a, b});
}
void fv_prof_end(int kind, cudaStream_t s) {
    std::lock_guard<std::mutex> lock(g_prof_mu);
    if (!g_prof_on || g_prof_ev[kind].empty()) return;
    cudaEventRecord(g_prof_ev[kind].back().second, s);
}

extern "C" {

int fv_profile(int32_t enable, double* ms, int64_t* launches) {
    std::lock_guard<std::mutex> lock(g_prof_mu);
    for (int k = 0; k < FV_K_COUNT; ++k) {
        double sum = 0.0;
        for (auto& pr : g_prof_ev[k]) {
            float t = 0.f;
            if (cudaEventSynchronize(pr.second) == cudaSuccess && cudaEventElapsedTime(&t, pr.first, pr.second) == cudaSuccess) sum += t;
            cudaEventDestroy(pr.first);
            cudaEventDestroy(pr.second);
        }
        if (ms) ms[k] = sum;
        if (launches) launches[k] = (int64_t)g_prof_ev[k].size();
        g_prof_ev[k].clear();
    }
    (void)cudaGetLastError();
    g_prof_on = enable != 0;
    return FV_OK;
}

const char* fv_last_error(void) { return g_err.c_str(); }
int64_t fv_launch_count(void) { return g_launches.load(); }
int64_t fv_n_weights(const fv_config* cfg) { return shape_ok(cfg) ? n_weights_of(cfg) : -1; }
int64_t fv_kv_bytes(const fv_model* m) { return m ? (int64_t)m->kv_bytes : 0; }
int32_t fv_kv_window(const fv_model* m) { return m ? m->window : 0; }

int fv_create_model(const fv_config* cfg, const float* weights, int64_t n_weights, const int32_t* mask_rowptr,
                    const int32_t* mask_col, const float* posemb, void* stream, fv_model** out) {
    if (!cfg || !weights || !mask_rowptr || !mask_col || !posemb || !out) return fail(FV_ERR_BAD_ARG, "null argument");
    if (!shape_ok(cfg)) return fail(FV_ERR_BAD_SHAPE, "unsupported d_model / n_heads / ffn_mult / act / n_layers");
    if (cfg->max_batch <= 0) return fail(FV_ERR_BAD_ARG, "max_batch must be positive");
    if (!(cfg->ln_eps > 0.f)) return fail(FV_ERR_BAD_ARG, "ln_eps must be positive");
    if (n_weights != n_weights_of(cfg)) return fail(FV_ERR_BAD_SHAPE, "n_weights does not match the configuration");
    const int N = cfg->n_sites, d = cfg->d_model, f = 4 * d, NL = cfg->n_layers;
    // mask validation (reading A11): ascending, unique, 0 <= col <= row, last entry == row
    if (mask_rowptr[0] != 0) return fail(FV_ERR_BAD_MASK, "rowptr[0] != 0");
    for (int t = 0; t < N; ++t)        // bound every row by rowptr[N] before any mask_col entry is read
        if (mask_rowptr[t + 1] <= mask_rowptr[t]) return fail(FV_ERR_BAD_MASK, "rowptr not increasing (empty mask row " + std::to_string(t) + ")");
    for (int t = 0; t < N; ++t) {
        const int e0 = mask_rowptr[t], e1 = mask_rowptr[t + 1];
        if (e1 <= e0) return fail(FV_ERR_BAD_MASK, "empty mask row " + std::to_string(t));
        for (int e = e0; e < e1; ++e) {
            if (mask_col[e] < 0 || mask_col[e] > t) return fail(FV_ERR_BAD_MASK, "col out of [0,row] in row " + std::to_string(t));
            if (e > e0 && mask_col[e] <= mask_col[e - 1]) return fail(FV_ERR_BAD_MASK, "row not ascending/unique: " + std::to_string(t));
        }
        if (mask_col[e1 - 1] != t) return fail(FV_ERR_BAD_MASK, "row must end with itself: " + std::to_string(t));
    }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDeviceProperties");
    if (prop.major != 10) return fail(FV_ERR_ARCH, "device is not compute capability 10.x (sm_100a required)");

    fv_model* m = new fv_model();
    m->cfg = *cfg;
    m->n_sms = prop.multiProcessorCount;
    m->mean_nnz = (double)mask_rowptr[N] / N;
    m->device = dev;
    Arena A;
    struct Off { size_t wqkv, wo, w1, w2, bqkv, bo, b1, b2, ln1g, ln1b, ln2g, ln2b, img_qkv, img_ffn, img_w1t, img_wo, par; };
    const bool lp_tc = d == 32 || d == 64 || d == 128;                     // fv_logprob.cu path
    const int KP = d < 64 ? 64 : d;
    const int HC = FV_LP_HC;
    std::vector<uint16_t> img((size_t)std::max(3 * d * KP, (f / HC) * (HC * KP + d * HC)));
    std::vector<Off> off(NL);
    const float* w = weights;
    const int V = cfg->vocab > 2 ? cfg->vocab : 2;
    const size_t o_tok = A.put(w, sizeof(float) * V * cfg->d_token);
    w += (size_t)V * cfg->d_token;
    std::vector<uint16_t> pk((size_t)f * d);
    std::vector<float> tmp((size_t)3 * d * d), tb(3 * d);
    for (int l = 0; l < NL; ++l) {
        Off& o = off[l];
        o.ln1g = A.put(w, 4 * d); w += d;
        o.ln1b = A.put(w, 4 * d); w += d;
        for (int p = 0; p < 3; ++p) {             // Wq,bq,Wk,bk,Wv,bv -> one [3d,d] matrix + [3d] bias
            std::memcpy(tmp.data() + (size_t)p * d * d, w, sizeof(float) * d * d); w += (size_t)d * d;
            std::memcpy(tb.data() + p * d, w, sizeof(float) * d); w += d;
        }
        pack_mma_a(tmp.data(), 3 * d, d, pk.data());
        o.wqkv = A.put(pk.data(), (size_t)3 * d * d * 2);
        o.img_qkv = o.img_ffn = o.img_w1t = 0;
        if (lp_tc) {
            fv_pack_sw128(tmp.data(), 3 * d, d, d, KP, img.data());
            o.img_qkv = A.put(img.data(), (size_t)3 * d * KP * 2);
        }
        o.bqkv = A.put(tb.data(), 4 * 3 * d);
        o.wo = o.bo = 0;
        o.img_wo = 0;
        if (cfg->has_wo) {
            if (lp_tc) {
                fv_pack_sw128(w, d, d, d, KP, img.data());
                o.img_wo = A.put(img.data(), (size_t)d * KP * 2);
            }
            pack_mma_a(w, d, d, pk.data()); w += (size_t)d * d;
            o.wo = A.put(pk.data(), (size_t)d * d * 2);
            o.bo = A.put(w, 4 * d); w += d;
        }
        o.ln2g = A.put(w, 4 * d); w += d;
        o.ln2b = A.put(w, 4 * d); w += d;
        pack_mma_a(w, f, d, pk.data());
        if (lp_tc) {                                  // per HC-column hidden chunk: W1_j | W2_j
            const float* W1 = w;
            const float* W2 = w + (size_t)f * d + f;   // after W1 and b1
            const size_t per = (size_t)HC * KP + (size_t)d * HC;
            for (int j = 0; j < f / HC; ++j) {
                fv_pack_sw128(W1 + (size_t)j * HC * d, HC, d, d, KP, img.data() + j * per);
                fv_pack_sw128(W2 + (size_t)j * HC, d, HC, f, HC, img.data() + j * per + (size_t)HC * KP);
            }
            o.img_ffn = A.put(img.data(), (size_t)(f / HC) * per * 2);
            o.img_w1t = 0;
            if (d == 128) {                           // fv_decode_tc.cu: the same W1 as [128 rows x 64 K] tiles, M-tile-major
                for (int mt = 0; mt < f / 128; ++mt) fv_pack_sw128(W1 + (size_t)mt * 128 * d, 128, d, d, d, img.data() + (size_t)mt * 128 * d);
                o.img_w1t = A.put(img.data(), (size_t)f * d * 2);
            }
        }
        w += (size_t)f * d;
        o.w1 = A.put(pk.data(), (size_t)f * d * 2);
        o.b1 = A.put(w, 4 * f); w += f;
        pack_mma_a(w, d, f, pk.data()); w += (size_t)d * f;
        o.w2 = A.put(pk.data(), (size_t)d * f * 2);
        o.b2 = A.put(w, 4 * d); w += d;
        {   // the same small parameters once more as one block (layout: fv_internal.h, FvLayerDev::par)
            std::vector<float> par((size_t)13 * d, 0.f);
            auto from = [&](size_t off, int n, int at) { std::memcpy(par.data() + at, A.host.data() + off, sizeof(float) * n); };
            from(o.ln1g, d, 0); from(o.ln1b, d, d); from(o.bqkv, 3 * d, 2 * d);
            from(o.ln2g, d, 5 * d); from(o.ln2b, d, 6 * d); from(o.b1, f, 7 * d); from(o.b2, d, 11 * d);
            if (cfg->has_wo) from(o.bo, d, 12 * d);
            o.par = A.put(par.data(), sizeof(float) * par.size());
        }
    }
    std::vector<float> wd(d);
    for (int i = 0; i < d; ++i) wd[i] = w[d + i] - w[i];            // head_W[1] - head_W[0]
    const float bd = w[(size_t)V * d + 1] - w[(size_t)V * d];
    const size_t o_wd = A.put(wd.data(), 4 * d);
    const size_t o_hw = A.put(w, sizeof(float) * (size_t)V * d);
    const size_t o_hb = A.put(w + (size_t)V * d, sizeof(float) * V);
    const size_t o_pos = A.put(posemb, sizeof(float) * (size_t)N * (d - cfg->d_token));
    const size_t o_rp = A.put(mask_rowptr, sizeof(int32_t) * (N + 1));
    const size_t o_col = A.put(mask_col, sizeof(int32_t) * (size_t)mask_rowptr[N]);
    // KV ring copy plan (fv_decode.cu): chunks of CH rows of A(t) \ {t}, runs of consecutive positions
    const int CH = fv_ring_ch(d);
    // Band mask (Eq. S1: M_ij = 0 iff i - j <= W): every row is the ONE run max(0, t-W)..t.  fv_sample then keeps
    // only a ring-buffer window of W+1 rows per (sample, layer): position p lives in row p % (W+1); the row step t appends
    // overwrites position t-W-1, which no later step attends.  FLASHVAN_KV=dense keeps the N-row pool (A/B measurements).
    int band_w = 0;
    for (int t = 0; t < N; ++t) band_w = std::max(band_w, t - mask_col[mask_rowptr[t]]);
    bool band = band_w >= 1 && 2 * (band_w + 1) <= N;
    for (int t = 0; t < N && band; ++t)
        band = mask_col[mask_rowptr[t]] == std::max(0, t - band_w) && mask_rowptr[t + 1] - mask_rowptr[t] == t - mask_col[mask_rowptr[t]] + 1;
    const bool band_shape = band;      // (the copy plans must not depend on the pool the environment picks)
    if (const char* kvm = std::getenv("FLASHVAN_KV"); kvm && std::strcmp(kvm, "dense") == 0) band = false;
    const int kv_rows = band ? band_w + 1 : N;
    m->window = band ? kv_rows : 0;
    std::vector<int32_t> chunk_ptr(N + 1, 0), chunk_run_ptr(1, 0);
    std::vector<int2> runs;
    for (int t = 0; t < N; ++t) {
        const int e0 = mask_rowptr[t], nn = mask_rowptr[t + 1] - 1 - e0;
        for (int c0 = 0; c0 < nn; c0 += CH) {
            const int rows = std::min(CH, nn - c0);
            for (int i = 0; i < rows;) {
                int j = i + 1;
                while (j < rows && mask_col[e0 + c0 + j] == mask_col[e0 + c0 + j - 1] + 1 &&
                       mask_col[e0 + c0 + j] % kv_rows != 0) ++j;          // a run ends where the window wraps
                runs.push_back(make_int2(mask_col[e0 + c0 + i] % kv_rows, (i << 16) | (j - i)));
                i = j;
            }
            chunk_run_ptr.push_back((int32_t)runs.size());
        }
        chunk_ptr[t + 1] = (int32_t)chunk_run_ptr.size() - 1;
    }
    if (runs.empty()) runs.push_back(make_int2(0, 0));
    // plan of fv_decode.cu (fv_internal.h: d_*): isolated positions first taken out, then the same chunking
    std::vector<int32_t> d_chunk_ptr(N + 1, 0), d_chunk_run_ptr(1, 0), d_nn(N, 0), d_dir((size_t)N * FV_DIRECT_MAX, -1);
    std::vector<int2> d_runs;
    for (int t = 0; t < N; ++t) {
        const int e0 = mask_rowptr[t], nn = mask_rowptr[t + 1] - 1 - e0;
        std::vector<int32_t> st;                                   // positions that stream through the ring
        int nd = 0;
        for (int i = 0; i < nn; ++i) {
            const int p0 = mask_col[e0 + i];
            const bool alone = (i == 0 || mask_col[e0 + i - 1] != p0 - 1) && (i + 1 == nn || mask_col[e0 + i + 1] != p0 + 1);
            if (alone && nd < FV_DIRECT_MAX && d <= 128 && !band_shape) d_dir[(size_t)t * FV_DIRECT_MAX + nd++] = p0 % kv_rows;
            else st.push_back(p0);
        }
        // a ragged tail of the ring's rows that still fits the direct slots goes the same way (cfg5: 65 = 4 x 16 + 1 rows:
        // no fifth chunk of one row per sample)
        if (const int rem = (int)st.size() % CH; rem > 0 && rem <= FV_DIRECT_MAX - nd && d <= 128 && !band_shape) {
            for (int i = 0; i < rem; ++i) d_dir[(size_t)t * FV_DIRECT_MAX + nd++] = st[st.size() - rem + i] % kv_rows;
            st.resize(st.size() - rem);
        }
        const int ns = (int)st.size();
        d_nn[t] = ns;
        for (int c0 = 0; c0 < ns; c0 += CH) {
            const int rows = std::min(CH, ns - c0);
            for (int i = 0; i < rows;) {
                int j = i + 1;
                while (j < rows && st[c0 + j] == st[c0 + j - 1] + 1 && st[c0 + j] % kv_rows != 0) ++j;
                d_runs.push_back(make_int2(st[c0 + i] % kv_rows, (i << 16) | (j - i)));
                i = j;
            }
            d_chunk_run_ptr.push_back((int32_t)d_runs.size());
        }
        d_chunk_ptr[t + 1] = (int32_t)d_chunk_run_ptr.size() - 1;
    }
    if (d_runs.empty()) d_runs.push_back(make_int2(0, 0));
    // block attention plan of fv_logprob.cu: union of the key positions of 32 consecutive mask rows
    const int BQ = 32;
    const int n_blk = (N + BQ - 1) / BQ;
    std::vector<int32_t> blk_uptr(1, 0), ukeys;
    std::vector<uint16_t> amask;
    for (int blk = 0; blk < n_blk; ++blk) {
        const int t0 = blk * BQ, t1 = std::min(N, t0 + BQ);
        std::vector<int32_t> u;
        for (int t = t0; t < t1; ++t) u.insert(u.end(), mask_col + mask_rowptr[t], mask_col + mask_rowptr[t + 1]);
        std::sort(u.begin(), u.end());
        u.erase(std::unique(u.begin(), u.end()), u.end());
        const size_t n_real = u.size();
        while (u.size() % 16) u.push_back(0);             // padding keys: a valid row, never allowed
        const size_t base = amask.size();
        amask.resize(base + u.size() / 16 * BQ, 0);
        for (int t = t0; t < t1; ++t)
            for (int e = mask_rowptr[t]; e < mask_rowptr[t + 1]; ++e) {
                const size_t k = std::lower_bound(u.begin(), u.begin() + n_real, mask_col[e]) - u.begin();
                amask[base + (k / 16) * BQ + (t - t0)] |= (uint16_t)(1u << (k % 16));
            }
        ukeys.insert(ukeys.end(), u.begin(), u.end());
        blk_uptr.push_back((int32_t)ukeys.size());
    }
    const size_t o_bu = A.put(blk_uptr.data(), sizeof(int32_t) * blk_uptr.size());
    const size_t o_uk = A.put(ukeys.data(), sizeof(int32_t) * ukeys.size());
    const size_t o_am = A.put(amask.data(), sizeof(uint16_t) * amask.size());
    const size_t o_cp = A.put(chunk_ptr.data(), sizeof(int32_t) * chunk_ptr.size());
    const size_t o_crp = A.put(chunk_run_ptr.data(), sizeof(int32_t) * chunk_run_ptr.size());
    const size_t o_runs = A.put(runs.data(), sizeof(int2) * runs.size());
    const size_t o_dcp = A.put(d_chunk_ptr.data(), sizeof(int32_t) * d_chunk_ptr.size());
    const size_t o_dcrp = A.put(d_chunk_run_ptr.data(), sizeof(int32_t) * d_chunk_run_ptr.size());
    const size_t o_druns = A.put(d_runs.data(), sizeof(int2) * d_runs.size());
    const size_t o_dnn = A.put(d_nn.data(), sizeof(int32_t) * d_nn.size());
    const size_t o_ddir = A.put(d_dir.data(), sizeof(int32_t) * d_dir.size());

    m->arena_bytes = A.host.size();
    e = cudaMalloc(&m->arena, m->arena_bytes);
    if (e != cudaSuccess) { delete m; return cuda_fail(e, "cudaMalloc(parameters)"); }
    m->kv_full_bytes = (size_t)cfg->max_batch * NL * N * 2 * d * sizeof(__nv_bfloat16);
    m->kv_bytes = (size_t)cfg->max_batch * NL * kv_rows * 2 * d * sizeof(__nv_bfloat16);
    void* kv = nullptr;
    e = cudaMalloc(&kv, m->kv_bytes);
    if (e != cudaSuccess) { cudaFree(m->arena); delete m; return cuda_fail(e, "cudaMalloc(KV pool)"); }
    if (lp_tc) {                                      // fv_log_prob workspace: h and q, fp32 [max_batch * N, d]
        m->ws_bytes = (size_t)2 * cfg->max_batch * N * d * sizeof(float);
        e = cudaMalloc(&m->ws, m->ws_bytes);
        if (e != cudaSuccess) { cudaFree(kv); cudaFree(m->arena); delete m; return cuda_fail(e, "cudaMalloc(log_prob workspace)"); }
    }
    if (const char* pz = std::getenv("FLASHVAN_POISON_KV"); pz && *pz == '1')   // debug aid: unwritten rows read as NaN
        cudaMemset(kv, 0xFF, m->kv_bytes);
    cudaStream_t s = (cudaStream_t)stream;
    e = cudaMemcpyAsync(m->arena, A.host.data(), m->arena_bytes, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { cudaFree(kv); cudaFree(m->ws); cudaFree(m->arena); delete m; return cuda_fail(e, "parameter upload"); }

    unsigned char* base = (unsigned char*)m->arena;
    FvModelDev& D = m->dev;
    D.n_sites = N; D.n_layers = NL; D.has_wo = cfg->has_wo; D.ln2_style = cfg->ln2_style;
    D.ln_eps = cfg->ln_eps; D.d_token = cfg->d_token;
    D.tok_emb = (const float*)(base + o_tok);
    D.posemb = (const float*)(base + o_pos);
    D.head_wd = (const float*)(base + o_wd);
    D.head_bd = bd;
    D.vocab = V;
    D.head_w = (const float*)(base + o_hw);
    D.head_b = (const float*)(base + o_hb);
    D.mask_rowptr = (const int32_t*)(base + o_rp);
    D.mask_col = (const int32_t*)(base + o_col);
    D.chunk_ptr = (const int32_t*)(base + o_cp);
    D.chunk_run_ptr = (const int32_t*)(base + o_crp);
    D.runs = (const int2*)(base + o_runs);
    D.d_chunk_ptr = (const int32_t*)(base + o_dcp);
    D.d_chunk_run_ptr = (const int32_t*)(base + o_dcrp);
    D.d_runs = (const int2*)(base + o_druns);
    D.d_nn = (const int32_t*)(base + o_dnn);
    D.d_dir = (const int32_t*)(base + o_ddir);
    D.att_blk_uptr = (const int32_t*)(base + o_bu);
    D.att_ukeys = (const int32_t*)(base + o_uk);
    D.att_mask = (const uint16_t*)(base + o_am);
    D.att_nblk = n_blk;
    D.kv_s = (__nv_bfloat16*)kv;
    D.kv_rows = kv_rows;
    D.kv = band ? nullptr : (__nv_bfloat16*)kv;       // window mode: fv_log_prob allocates its N-row pool at its first call
    D.lp_h = (float*)m->ws;
    D.lp_q = m->ws ? (float*)m->ws + (size_t)cfg->max_batch * N * d : nullptr;
    for (int l = 0; l < NL; ++l) {
        const Off& o = off[l];
        FvLayerDev& L = D.layer[l];
        L.wqkv = (const uint4*)(base + o.wqkv);
        L.wo = cfg->has_wo ? (const uint4*)(base + o.wo) : nullptr;
        L.w1 = (const uint4*)(base + o.w1);
        L.w2 = (const uint4*)(base + o.w2);
        L.bqkv = (const float*)(base + o.bqkv);
        L.bo = cfg->has_wo ? (const float*)(base + o.bo) : nullptr;
        L.b1 = (const float*)(base + o.b1);
        L.b2 = (const float*)(base + o.b2);
        L.ln1_g = (const float*)(base + o.ln1g); L.ln1_b = (const float*)(base + o.ln1b);
        L.ln2_g = (const float*)(base + o.ln2g); L.ln2_b = (const float*)(base + o.ln2b);
        L.par = (const float*)(base + o.par);
        L.img_qkv = lp_tc ? base + o.img_qkv : nullptr;
        L.img_ffn = lp_tc ? base + o.img_ffn : nullptr;
        L.img_w1t = (lp_tc && d == 128 && !cfg->has_wo) ? base + o.img_w1t : nullptr;
        L.img_wo = (lp_tc && cfg->has_wo) ? base + o.img_wo : nullptr;
    }
    *out = m;
    return FV_OK;
}

void fv_destroy_model(fv_model* m) {
    if (!m) return;
    int cur = -1;
    cudaGetDevice(&cur);
    if (cur != m->device) cudaSetDevice(m->device);      // free on the model's own device, then restore
    cudaDeviceSynchronize();
    if (m->dev.kv != m->dev.kv_s) cudaFree(m->dev.kv);
    cudaFree(m->dev.kv_s);
    cudaFree(m->ws);
    cudaFree(m->arena);
    if (cur >= 0 && cur != m->device) cudaSetDevice(cur);
    delete m;
}

// Ordered Markov boundary -> mask rows (fv_mask.cu does the graph work).
int fv_markov_mask(int32_t n, int64_t n_edges, const int32_t* edge_a, const int32_t* edge_b,
                   int32_t position_space, int32_t* out_rowptr, int32_t* out_col, int64_t cap,
                   int64_t* nnz, int32_t* d_max) {
    if (n <= 0 || n_edges < 0 || (n_edges > 0 && (!edge_a || !edge_b)) || !out_rowptr || cap < 0 ||
        (cap > 0 && !out_col) || (position_space != 0 && position_space != 1))
        return fail(FV_ERR_BAD_ARG, "fv_markov_mask: bad argument");
    std::vector<std::vector<int32_t>> rows;
    std::string err;
    if (fv_markov_rows(n, n_edges, edge_a, edge_b, rows, err) != 0) return fail(FV_ERR_BAD_ARG, "fv_markov_mask: " + err);
    int64_t total = 0;
    int32_t dm = 0;
    for (int32_t i = 0; i < n; ++i) {
        const std::vector<int32_t>& r = rows[i];
        if (!r.empty()) dm = std::max(dm, i - r.front());
        // position space: j + 1 for every boundary vertex, and t itself exactly once
        total += position_space ? (int64_t)r.size() + ((!r.empty() && r.back() == i - 1) ? 0 : 1) : (int64_t)r.size();
    }
    if (nnz) *nnz = total;
    if (d_max) *d_max = dm;
    if (total > 0x7fffffffLL) return fail(FV_ERR_BAD_SHAPE, "fv_markov_mask: more than 2^31 - 1 mask entries");
    int64_t at = 0;
    out_rowptr[0] = 0;
    for (int32_t i = 0; i < n; ++i) {
        const std::vector<int32_t>& r = rows[i];
        const int64_t len = position_space ? (int64_t)r.size() + ((!r.empty() && r.back() == i - 1) ? 0 : 1) : (int64_t)r.size();
        if (total <= cap) {
            for (int32_t j : r)
                if (!position_space) out_col[at++] = j;
                else if (j + 1 < i) out_col[at++] = j + 1;
            if (position_space) out_col[at++] = i;
        }
        out_rowptr[i + 1] = (int32_t)(out_rowptr[i] + len);
    }
    if (total > cap) return fail(FV_ERR_BAD_ARG, "fv_markov_mask: out_col holds " + std::to_string(cap) + " entries, " + std::to_string(total) + " needed");
    return FV_OK;
}

// Launch geometry of the persistent forward kernel.
// SAMPLE: one CTA per SM; B samples are cut into groups of S <= 32 so that the number of groups
// is (a multiple of) the SM count; NT = ceil(S/8) rounded to {1,2,4} n8-tiles per mma.
static void sample_geometry(int B, int n_sms, int* S, int* nt, int* n_groups, int* grid) {
    const int rounds = (B + n_sms * 32 - 1) / (n_sms * 32);
    const int target = rounds * n_sms;
    int s = (B + target - 1) / target;
    if (s < 1) s = 1;
    *nt = s <= 8 ? 1 : (s <= 16 ? 2 : 4);
    *S = s;
    *n_groups = (B + s - 1) / s;
    *grid = *n_groups < n_sms ? *n_groups : n_sms;
}

int fv_sample(fv_model* m, int32_t B, const float* uniforms, int8_t* spins, float* logq, float* cond_p,
              void* stream) {
    if (!m || !uniforms || !spins || !logq) return fail(FV_ERR_BAD_ARG, "null argument");
    if (B <= 0 || B > m->cfg.max_batch) return fail(FV_ERR_BAD_ARG, "B must be in [1, max_batch]");
    if (int rc = wrong_device(m)) return rc;
    FvForwardArgs a{};
    a.mode = FV_MODE_SAMPLE;
    a.B = B;
    int nt, grid;
    sample_geometry(B, m->n_sms, &a.rows_per_group, &nt, &a.n_groups, &grid);
    a.uniforms = uniforms; a.spins_out = spins; a.logq = logq; a.cond_p = cond_p;
    (void)grid;
    // Two samplers.  Default for d = 128 models with short mask rows (the per-step cost is latency, not KV bytes):
    // the layer-pipelined clusters of fv_chain.cu with the weights resident in tensor / shared memory; otherwise
    // (and for every other shape) the streaming kernel of fv_decode.cu.  FLASHVAN_DECODE=chain | ring forces one.
    const char* dmode = std::getenv("FLASHVAN_DECODE");
    const bool force_chain = dmode && std::strcmp(dmode, "chain") == 0;
    if (wants_chain(m)) {
        fv_prof_begin(FV_K_SAMPLE, (cudaStream_t)stream);
        cudaError_t ec = fv_launch_chain(m->dev, m->cfg.d_model, m->cfg.d_model / m->cfg.n_heads, a, (cudaStream_t)stream);
        fv_prof_end(FV_K_SAMPLE, (cudaStream_t)stream);
        if (ec == cudaSuccess) { g_launches++; return FV_OK; }
        if (ec != cudaErrorNotSupported) return cuda_fail(ec, "fv_sample launch (chain)");
        (void)cudaGetLastError();
        if (force_chain) return fail(FV_ERR_BAD_SHAPE, "FLASHVAN_DECODE=chain: shape not covered by the chain sampler");
    }
    // FLASHVAN_DECODE=cluster opts into the 2-CTA-cluster FFN split (correct, but measured slower than one
    // CTA per sample group on every BASELINE config: DESIGN.md 6.1)
    const char* dm = std::getenv("FLASHVAN_DECODE");
    const int cluster = dm && std::strcmp(dm, "cluster") == 0 && !m->cfg.has_wo;
    fv_prof_begin(FV_K_SAMPLE, (cudaStream_t)stream);
    cudaError_t e = cudaErrorNotSupported;
    if (wants_tc(m, nt)) e = fv_launch_decode_tc(m->dev, m->cfg.d_model, m->cfg.d_model / m->cfg.n_heads, nt, a, m->n_sms, (cudaStream_t)stream);
    if (e == cudaErrorNotSupported) {
        (void)cudaGetLastError();
        e = fv_launch_decode(m->dev, m->cfg.d_model, m->cfg.d_model / m->cfg.n_heads, nt, a, m->n_sms, cluster, (cudaStream_t)stream);
    }
    fv_prof_end(FV_K_SAMPLE, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "fv_sample launch");
    g_launches++;
    return FV_OK;
}

const char* fv_sampler_kind(const fv_model* m, int32_t B) {
    if (!m || B <= 0) return "none";
    if (wants_chain(m) && fv_chain_supported(m->dev, m->cfg.d_model, m->cfg.d_model / m->cfg.n_heads, B)) return "chain";
    int S, nt, ng, grid;
    sample_geometry(B, m->n_sms, &S, &nt, &ng, &grid);
    return wants_tc(m, nt) && m->cfg.d_model == 128 && m->cfg.d_model / m->cfg.n_heads == 16 && !m->cfg.has_wo ? "ring-tc" : "ring";
}

int fv_log_prob(fv_model* m, int32_t B, const int8_t* spins, float* logq, float* cond_p, void* stream) {
    if (!m || !spins || !logq) return fail(FV_ERR_BAD_ARG, "null argument");
    if (B <= 0 || B > m->cfg.max_batch) return fail(FV_ERR_BAD_ARG, "B must be in [1, max_batch]");
    if (int rc = wrong_device(m)) return rc;
    if (!m->dev.kv) {                                              // window mode: the teacher-forced pass needs all N rows
        void* kv = nullptr;
        cudaError_t ea = cudaMalloc(&kv, m->kv_full_bytes);
        if (ea != cudaSuccess) return cuda_fail(ea, "cudaMalloc(fv_log_prob KV pool)");
        m->dev.kv = (__nv_bfloat16*)kv;
    }
    const char* force = std::getenv("FLASHVAN_LOGPROB");          // "chunked": the persistent teacher-forcing kernel
    if (m->dev.vocab > 2) force = nullptr;                         // (one spin per token only)
    if (!(force && std::strcmp(force, "chunked") == 0)) {
        int n_launch = 0;
        cudaError_t e2 = fv_launch_logprob_tc(m->dev, m->cfg.d_model, m->cfg.d_model / m->cfg.n_heads, B, spins, logq,
                                              cond_p, m->n_sms, &n_launch, (cudaStream_t)stream);
        if (e2 == cudaSuccess) { g_launches += n_launch; return FV_OK; }
        if (e2 != cudaErrorNotSupported) return cuda_fail(e2, "fv_log_prob launch");
        (void)cudaGetLastError();
    }
    FvForwardArgs a{};
    a.mode = FV_MODE_LOGPROB;
    a.B = B;
    a.samples_per_cta = (B + m->n_sms - 1) / m->n_sms;
    const int grid = (B + a.samples_per_cta - 1) / a.samples_per_cta;
    a.spins_in = spins; a.logq = logq; a.cond_p = cond_p;
    // small tiles when a CTA owns very few rows, else 32-row tiles (least weight traffic per row)
    const long long rows = (long long)a.samples_per_cta * m->cfg.n_sites;
    const int nt = rows <= 8 ? 1 : (rows <= 16 ? 2 : 4);
    cudaError_t e = fv_launch_forward(m->dev, m->cfg.d_model, m->cfg.d_model / m->cfg.n_heads, nt, a, grid,
                                      (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "fv_log_prob launch");
    g_launches++;
    return FV_OK;
}

static_assert(FV_LP_STATIC_BYTES == FV_STATIC_SCRATCH_BYTES, "flashvan.h and fv_internal.h disagree on the static scratch size");

int fv_log_prob_static(fv_model* m, int32_t B, const int8_t* spins, float* logq, float* cond_p, void* stream) {
    if (!m || !spins || !logq) return fail(FV_ERR_BAD_ARG, "null argument");
    if (B <= 0) return fail(FV_ERR_BAD_ARG, "B must be positive");
    if (int rc = wrong_device(m)) return rc;
    if (m->cfg.d_model > 128)
        return fail(FV_ERR_BAD_SHAPE, "fv_log_prob_static: only the layer-major path (d_model <= 128)");
    const size_t need = fv_logprob_static_need(m->dev, m->cfg.d_model, B);
    if (need > FV_LP_STATIC_BYTES)
        return fail(FV_ERR_BAD_ARG, "fv_log_prob_static: B * N = " + std::to_string((long long)B * m->cfg.n_sites) + " rows need " +
                                        std::to_string(need) + " bytes of workspace, the static array holds " +
                                        std::to_string(FV_LP_STATIC_BYTES) + " (use fv_log_prob)");
    int n_launch = 0;
    cudaError_t e = fv_launch_logprob_tc_static(m->dev, m->cfg.d_model, m->cfg.d_model / m->cfg.n_heads, B, spins, logq, cond_p,
                                                m->n_sms, &n_launch, (cudaStream_t)stream);
    if (e == cudaErrorNotSupported) { (void)cudaGetLastError(); return fail(FV_ERR_BAD_SHAPE, "fv_log_prob_static: shape not covered by the layer-major path"); }
    if (e != cudaSuccess) return cuda_fail(e, "fv_log_prob_static launch");
    g_launches += n_launch;
    return FV_OK;
}

int fv_energy_csr(int32_t B, int32_t N, const int8_t* spins, const int32_t* rowptr, const int32_t* col,
                  const float* val, int32_t integer_couplings, float* E, void* stream) {
    if (!spins || !rowptr || !col || !val || !E) return fail(FV_ERR_BAD_ARG, "null argument");
    if (B <= 0 || N <= 0) return fail(FV_ERR_BAD_ARG, "B and N must be positive");
    cudaError_t e = fv_launch_energy_csr(B, N, spins, rowptr, col, val, integer_couplings, E, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "fv_energy_csr launch");
    g_launches++;
    return FV_OK;
}

int fv_energy_dense(int32_t B, int32_t N, const int8_t* spins, const float* J, float* E, void* stream) {
    if (!spins || !J || !E) return fail(FV_ERR_BAD_ARG, "null argument");
    if (B <= 0 || N <= 0) return fail(FV_ERR_BAD_ARG, "B and N must be positive");
    cudaError_t e = fv_launch_energy_dense(B, N, spins, J, E, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "fv_energy_dense launch");
    g_launches++;
    return FV_OK;
}

int fv_free_energy(int32_t B, const float* E, const float* logq, double temperature, double* out, void* stream) {
    if (!E || !logq || !out) return fail(FV_ERR_BAD_ARG, "null argument");
    if (B <= 0) return fail(FV_ERR_BAD_ARG, "B must be positive");
    cudaError_t e = fv_launch_free_energy(B, E, logq, temperature, out, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "fv_free_energy launch");
    g_launches++;
    return FV_OK;
}

int fv_tokens_to_spins(int32_t B, int32_t n_tokens, int32_t P, const uint8_t* tokens, const int32_t* site_index,
                       int8_t* spins, void* stream) {
    if (!tokens || !site_index || !spins) return fail(FV_ERR_BAD_ARG, "null argument");
    if (B <= 0 || n_tokens <= 0 || P <= 0 || P > 8) return fail(FV_ERR_BAD_ARG, "B, n_tokens must be positive and 1 <= P <= 8");
    cudaError_t e = fv_launch_tokens_to_spins(B, n_tokens, P, tokens, site_index, spins, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "fv_tokens_to_spins launch");
    g_launches++;
    return FV_OK;
}

int fv_overlap(int32_t B, int32_t N, const int8_t* spins_a, const int8_t* spins_b, int32_t* dot, int32_t* hist,
               void* stream) {
    if (!spins_a || !spins_b || !dot) return fail(FV_ERR_BAD_ARG, "null argument");
    if (B <= 0 || N <= 0) return fail(FV_ERR_BAD_ARG, "B and N must be positive");
    cudaError_t e = fv_launch_overlap(B, N, spins_a, spins_b, dot, hist, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "fv_overlap launch");
    g_launches++;
    return FV_OK;
}

int fv_lmc_sweeps(int32_t B, int32_t N, int32_t n_sweeps, int8_t* spins, const int32_t* adj_rowptr,
                  const int32_t* adj_col, const float* adj_val, float beta, const float* exp_variates,
                  int32_t* accepted, void* stream) {
    if (B <= 0 || N <= 0 || n_sweeps < 0) return fail(FV_ERR_BAD_ARG, "B, N must be positive and n_sweeps >= 0");
    if (!spins || !adj_rowptr || !adj_col || !adj_val || (n_sweeps > 0 && !exp_variates)) return fail(FV_ERR_BAD_ARG, "null argument");
    if (N > 48 * 1024) return fail(FV_ERR_BAD_SHAPE, "fv_lmc_sweeps keeps a sample's spins in shared memory: N <= 49152");
    cudaError_t e = fv_launch_lmc(B, N, n_sweeps, spins, adj_rowptr, adj_col, adj_val, beta, exp_variates, accepted,
                                  (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "fv_lmc_sweeps launch");
    g_launches++;
    return FV_OK;
}

}  // extern "C"
