// fv_forward.cu -- the persistent FlashVAN forward kernel for sm_100a.
//
// One kernel serves both execution modes of the paper's network:
//   SAMPLE  (Alg. 2): a CTA owns a group of S <= 8*NT samples for all N
//           steps; a "tile" is those S samples at one position t.
//   LOGPROB (Alg. 1): a CTA owns whole samples and walks their positions in
//           ascending order, 8*NT consecutive positions per tile (chunked teacher forcing).
// In both modes a tile goes through embed -> n_l x [LN1, QKV, KV append, masked gather
// attention, (W_O), LN2, FFN] -> head, and attention reads only the KV rows named by the CSR
// mask row of its position from the bf16 KV pool, so no N x N score matrix ever exists.
// CTAs never communicate: samples are independent, so no grid-wide sync.
//
// GEMMs (this revision): weights are the 16-row "A" operand of mma.sync.m16n8k16 (bf16 in,
// fp32 accumulate), streamed straight from L2 in pre-packed fragment order (one coalesced
// 512 B warp load per 16x16 tile); the tile's rows are the n8 operand read from shared
// memory.  With 7-32 rows per CTA these projections are bound by the L2->SM weight stream,
// not by tensor throughput.
#include "fv_device.cuh"

namespace {
using namespace fvdev;

template <int D, int DH, int NT, int NW>
__global__ void __launch_bounds__(NW * 32, 1)
fv_forward_kernel(const __grid_constant__ FvModelDev m, const __grid_constant__ FvForwardArgs a) {
    using G = Geo<D, NT>;
    constexpr int R = G::R, HS = G::HS, AS = G::AS, QS = G::QS, FS = G::FS, KS2 = G::KS2;
    constexpr int NSPLIT = (NW / R) > 1 ? (NW / R) : 1;     // warps cooperating on one query row
    constexpr int LPR = D / 8, RPI = 32 / LPR;
    constexpr int SPS = D + 2 * LPR;                         // floats per split-partial slot
    static_assert(R * NSPLIT <= 16 || NSPLIT == 1, "split slots");

    extern __shared__ __align__(16) unsigned char smem[];
    float* sh_h = reinterpret_cast<float*>(smem);
    __nv_bfloat16* sh_a = reinterpret_cast<__nv_bfloat16*>(smem + G::h_bytes);
    unsigned char* big = smem + G::h_bytes + G::a_bytes;
    float* sh_qkv = reinterpret_cast<float*>(big);
    __nv_bfloat16* sh_hid = reinterpret_cast<__nv_bfloat16*>(big);
    float* sh_part = reinterpret_cast<float*>(big + G::hid_bytes);
    float* sh_split = reinterpret_cast<float*>(big + G::big_bytes);
    double* sh_logq = reinterpret_cast<double*>(big + G::big_bytes + G::split_bytes);
    float* sh_logp = reinterpret_cast<float*>(sh_logq + R);
    float* sh_u = sh_logp + R;
    int* sh_tok = reinterpret_cast<int*>(sh_u + R);
    int* sh_b = sh_tok + R;       // sample index of the row, -1 if the row is padding
    int* sh_t = sh_b + R;         // position of the row

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = lane >> 2, c = lane & 3;
    const int N = m.n_sites, NL = m.n_layers;
    const bool sample_mode = (a.mode == FV_MODE_SAMPLE);

    // work assignment
    int unit = blockIdx.x, unit_end, unit_step;
    int b_first = 0, n_own = 0, n_tiles = 0;
    if (sample_mode) { unit_end = a.n_groups; unit_step = gridDim.x; }
    else { unit_end = unit + 1; unit_step = 1; }
    double lq_carry = 0.0;                                   // LOGPROB: thread 0 only

    for (; unit < unit_end; unit += unit_step) {
        if (sample_mode) {
            b_first = unit * a.rows_per_group;
            n_own = min(a.rows_per_group, a.B - b_first);
            n_tiles = N;
            if (tid < R) { sh_tok[tid] = 0; sh_logq[tid] = 0.0; }
        } else {
            b_first = unit * a.samples_per_cta;
            n_own = min(a.samples_per_cta, a.B - b_first);
            if (n_own <= 0) return;
            n_tiles = (int)(((long long)n_own * N + R - 1) / R);
        }
        for (int tile = 0; tile < n_tiles; ++tile) {
            // ---- row descriptors -------------------------------------------------------
            if (tid < R) {
                int b, t, tok;
                if (sample_mode) {
                    b = tid < n_own ? b_first + tid : -1;
                    t = tile;
                    tok = sh_tok[tid];
                    sh_u[tid] = b >= 0 ? __ldg(a.uniforms + (size_t)b * N + t) : 2.f;
                } else {
                    const long long gi = (long long)tile * R + tid;
                    const bool ok = gi < (long long)n_own * N;
                    b = ok ? b_first + (int)(gi / N) : -1;
                    t = ok ? (int)(gi % N) : 0;
                    tok = (ok && t > 0) ? (a.spins_in[(size_t)b * N + t - 1] > 0 ? 1 : 0) : 0;
                    sh_tok[tid] = tok;
                }
                sh_b[tid] = b;
                sh_t[tid] = t;
            }
            __syncthreads();
            // ---- concatenated positional embedding (Eq. 15, l.287-292) -------------------
            for (int i = tid; i < R * D; i += NW * 32) {
                const int r = i / D, f = i - r * D;
                const int dt = m.d_token;
                sh_h[r * HS + f] = f < dt ? __ldg(m.tok_emb + sh_tok[r] * dt + f)
                                          : __ldg(m.posemb + (size_t)sh_t[r] * (D - dt) + (f - dt));
            }
            __syncthreads();
            for (int l = 0; l < NL; ++l) {
                const FvLayerDev& L = m.layer[l];
                // ---- LN1 (Alg. 2 l.12) -> bf16 activations ----------------------------------
                for (int r = warp; r < R; r += NW)
                    ln_row<D>(sh_h + r * HS, L.ln1_g, L.ln1_b, m.ln_eps, false, sh_a + r * AS, lane);
                __syncthreads();
                // ---- q, k, v = W a + b (Eq. 2; Alg. 2 l.13) ---------------------------------
                gemm_rows<D / 16, 1, NT, NW>(L.wqkv, 3 * D / 16, sh_a, AS, warp, lane,
                    [&](int mt, int, float (&acc)[NT][4]) {
                        const int f = mt * 16 + g;
                        const float b0 = __ldg(L.bqkv + f), b1 = __ldg(L.bqkv + f + 8);
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) {
                            float* o = sh_qkv + (nt * 8 + 2 * c) * QS + f;
                            o[0] = acc[nt][0] + b0; o[QS] = acc[nt][1] + b0;
                            o[8] = acc[nt][2] + b1; o[QS + 8] = acc[nt][3] + b1;
                        }
                    });
                __syncthreads();
                // ---- append k_t, v_t to the KV pool as bf16 (Alg. 2 l.17; reading A2: before
                //      the attention, so position t attends itself) --------------------------
                for (int i = tid; i < R * (2 * D / 8); i += NW * 32) {
                    const int r = i / (2 * D / 8), ch = i - r * (2 * D / 8);
                    const int b = sh_b[r];
                    if (b < 0) continue;
                    const float* s = sh_qkv + r * QS + D + ch * 8;
                    uint4 v;
                    v.x = pack_bf16(s[0], s[1]); v.y = pack_bf16(s[2], s[3]);
                    v.z = pack_bf16(s[4], s[5]); v.w = pack_bf16(s[6], s[7]);
                    __nv_bfloat16* dst = m.kv + (((size_t)b * NL + l) * N + sh_t[r]) * (2 * D) + ch * 8;
                    *reinterpret_cast<uint4*>(dst) = v;
                }
                __syncthreads();
                // ---- masked gather attention + residual (Eq. 3; Alg. 2 l.14-15) -------------
                for (int task = warp; task < R * NSPLIT; task += NW) {
                    const int r = task / NSPLIT, sp = task - r * NSPLIT;
                    const int b = sh_b[r];
                    if (b < 0) continue;
                    const int t = sh_t[r];
                    int e0 = __ldg(m.mask_rowptr + t), e1 = __ldg(m.mask_rowptr + t + 1);
                    if (NSPLIT > 1) {
                        int chunk = (e1 - e0 + NSPLIT - 1) / NSPLIT;
                        chunk = (chunk + RPI - 1) / RPI * RPI;
                        e0 = min(e0 + sp * chunk, e1);
                        e1 = min(e0 + chunk, e1);
                    }
                    float mm, ll, acc[8];
                    attend_range<D, DH>(sh_qkv + r * QS, m.kv + ((size_t)b * NL + l) * N * (2 * D), m.mask_col,
                                        e0, e1, lane, mm, ll, acc);
                    if (lane < LPR) {
                        if (NSPLIT > 1) {
                            float* ps = sh_split + task * SPS;
                            ps[lane] = mm; ps[LPR + lane] = ll;
#pragma unroll
                            for (int j = 0; j < 8; ++j) ps[2 * LPR + lane * 8 + j] = acc[j];
                        } else {
                            const float inv = 1.0f / ll;
                            if (m.has_wo) {
#pragma unroll
                                for (int j = 0; j < 8; ++j) sh_a[r * AS + lane * 8 + j] = __float2bfloat16_rn(acc[j] * inv);
                            } else {
#pragma unroll
                                for (int j = 0; j < 8; ++j) sh_h[r * HS + lane * 8 + j] += acc[j] * inv;
                            }
                        }
                    }
                }
                __syncthreads();
                if (NSPLIT > 1) {                       // combine the split partials, fixed order
                    for (int i = tid; i < R * D; i += NW * 32) {
                        const int r = i / D, f = i - r * D;
                        if (sh_b[r] < 0) continue;
                        const float* ps = sh_split + r * NSPLIT * SPS;
                        float mx = -1e30f;
#pragma unroll
                        for (int s = 0; s < NSPLIT; ++s) mx = fmaxf(mx, ps[s * SPS + f / 8]);
                        float num = 0.f, den = 0.f;
#pragma unroll
                        for (int s = 0; s < NSPLIT; ++s) {
                            const float w = fast_exp2(ps[s * SPS + f / 8] - mx);
                            den += w * ps[s * SPS + LPR + f / 8];
                            num += w * ps[s * SPS + 2 * LPR + f];
                        }
                        const float u = num / den;
                        if (m.has_wo) sh_a[r * AS + f] = __float2bfloat16_rn(u);
                        else sh_h[r * HS + f] += u;
                    }
                    __syncthreads();
                }
                // ---- optional output projection (bypassed in the paper, l.107) --------------
                if (m.has_wo) {
                    gemm_rows<D / 16, 1, NT, NW>(L.wo, D / 16, sh_a, AS, warp, lane,
                        [&](int mt, int, float (&acc)[NT][4]) {
                            const int f = mt * 16 + g;
                            const float b0 = __ldg(L.bo + f), b1 = __ldg(L.bo + f + 8);
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt) {
                                float* o = sh_h + (nt * 8 + 2 * c) * HS + f;
                                o[0] += acc[nt][0] + b0; o[HS] += acc[nt][1] + b0;
                                o[8] += acc[nt][2] + b1; o[HS + 8] += acc[nt][3] + b1;
                            }
                        });
                    __syncthreads();
                }
                // ---- LN2 (Alg. 2 l.16; ln2_style 1 = Alg. 1 l.5) ----------------------------
                for (int r = warp; r < R; r += NW)
                    ln_row<D>(sh_h + r * HS, L.ln2_g, L.ln2_b, m.ln_eps, m.ln2_style == 1, sh_a + r * AS, lane);
                __syncthreads();
                // ---- FFN up-projection + exact GELU -> bf16 hidden ---------------------------
                gemm_rows<D / 16, 1, NT, NW>(L.w1, 4 * D / 16, sh_a, AS, warp, lane,
                    [&](int mt, int, float (&acc)[NT][4]) {
                        const int f = mt * 16 + g;
                        const float b0 = __ldg(L.b1 + f), b1 = __ldg(L.b1 + f + 8);
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) {
                            __nv_bfloat16* o = sh_hid + (nt * 8 + 2 * c) * FS + f;
                            o[0] = __float2bfloat16_rn(gelu_erf(acc[nt][0] + b0));
                            o[FS] = __float2bfloat16_rn(gelu_erf(acc[nt][1] + b0));
                            o[8] = __float2bfloat16_rn(gelu_erf(acc[nt][2] + b1));
                            o[FS + 8] = __float2bfloat16_rn(gelu_erf(acc[nt][3] + b1));
                        }
                    });
                __syncthreads();
                // ---- FFN down-projection, K split KS2 ways into partial buffers -------------
                gemm_rows<4 * D / 16, KS2, NT, NW>(L.w2, D / 16, sh_hid, FS, warp, lane,
                    [&](int mt, int ks, float (&acc)[NT][4]) {
                        const int f = mt * 16 + g;
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) {
                            float* o = sh_part + ((size_t)ks * R + nt * 8 + 2 * c) * HS + f;
                            o[0] = acc[nt][0]; o[HS] = acc[nt][1];
                            o[8] = acc[nt][2]; o[HS + 8] = acc[nt][3];
                        }
                    });
                __syncthreads();
                // ---- feed-forward residual (Alg. 2 l.16) ------------------------------------
                for (int i = tid; i < R * D; i += NW * 32) {
                    const int r = i / D, f = i - r * D;
                    float v = __ldg(L.b2 + f);
#pragma unroll
                    for (int ks = 0; ks < KS2; ++ks) v += sh_part[((size_t)ks * R + r) * HS + f];
                    sh_h[r * HS + f] += v;
                }
                __syncthreads();
            }
            // ---- output head: p(+1) = softmax(z)[1] = sigmoid(z1 - z0) (Alg. 2 l.20-22) -----
            for (int r = warp; r < R; r += NW) {
                const int b = sh_b[r];
                if (b < 0) continue;
                float d = 0.f;
#pragma unroll
                for (int j = 0; j < D / 32; ++j) d += sh_h[r * HS + lane * (D / 32) + j] * __ldg(m.head_wd + lane * (D / 32) + j);
                d = warp_sum(d) + m.head_bd;
                if (lane == 0) {
                    const int t = sh_t[r];
                    const float p = 1.0f / (1.0f + expf(-d));
                    int up;
                    if (sample_mode) {
                        up = sh_u[r] < p;                               // reading A10 (l.23)
                        a.spins_out[(size_t)b * N + t] = up ? 1 : -1;    // sigma = 2 s - 1 (l.25)
                        sh_tok[r] = up;
                    } else {
                        up = a.spins_in[(size_t)b * N + t] > 0;
                    }
                    const float x = up ? -d : d;                        // log p(s) = -softplus(x)
                    sh_logp[r] = -(fmaxf(x, 0.f) + log1pf(expf(-fabsf(x))));
                    if (a.cond_p) a.cond_p[(size_t)b * N + t] = p;
                }
            }
            __syncthreads();
            // ---- log q accumulation in fp64, fixed order (Alg. 1 l.9) --------------------------
            if (sample_mode) {
                if (tid < n_own) {
                    sh_logq[tid] += (double)sh_logp[tid];
                    if (tile == N - 1) a.logq[b_first + tid] = (float)sh_logq[tid];
                }
            } else if (tid == 0) {
                for (int r = 0; r < R; ++r) {
                    if (sh_b[r] < 0) break;
                    if (sh_t[r] == 0) lq_carry = 0.0;
                    lq_carry += (double)sh_logp[r];
                    if (sh_t[r] == N - 1) a.logq[sh_b[r]] = (float)lq_carry;
                }
            }
            __syncthreads();
        }
    }
}

}  // namespace

// ------------------------------------------------------------------------------ dispatch
template <int D, int DH, int NT>
static cudaError_t launch_one(const FvModelDev& m, const FvForwardArgs& a, int grid, cudaStream_t s) {
    constexpr int NW = 16;
    auto kern = fv_forward_kernel<D, DH, NT, NW>;
    const size_t smem = Geo<D, NT>::total;
    if (cudaError_t e = fv_smem_attr((const void*)kern, (int)smem); e != cudaSuccess) return e;
    kern<<<grid, NW * 32, smem, s>>>(m, a);
    return cudaGetLastError();
}

template <int D, int DH>
static cudaError_t launch_nt(const FvModelDev& m, int nt, const FvForwardArgs& a, int grid, cudaStream_t s) {
    switch (nt) {
        case 1: return launch_one<D, DH, 1>(m, a, grid, s);
        case 2: return launch_one<D, DH, 2>(m, a, grid, s);
        case 4: return launch_one<D, DH, 4>(m, a, grid, s);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t fv_launch_forward(const FvModelDev& m, int d_model, int d_head, int nt, const FvForwardArgs& a,
                              int grid, cudaStream_t s) {
    const int key = d_model * 1000 + d_head;
    switch (key) {
        case 32016: return launch_nt<32, 16>(m, nt, a, grid, s);
        case 64016: return launch_nt<64, 16>(m, nt, a, grid, s);
        case 64032: return launch_nt<64, 32>(m, nt, a, grid, s);
        case 128016: return launch_nt<128, 16>(m, nt, a, grid, s);
        case 128032: return launch_nt<128, 32>(m, nt, a, grid, s);
        case 256064: return launch_nt<256, 64>(m, nt, a, grid, s);
        default: return cudaErrorInvalidValue;
    }
}

size_t fv_forward_smem_bytes(int d_model, int nt) {
    switch (d_model * 10 + nt) {
        case 321: return Geo<32, 1>::total;   case 322: return Geo<32, 2>::total;   case 324: return Geo<32, 4>::total;
        case 641: return Geo<64, 1>::total;   case 642: return Geo<64, 2>::total;   case 644: return Geo<64, 4>::total;
        case 1281: return Geo<128, 1>::total; case 1282: return Geo<128, 2>::total; case 1284: return Geo<128, 4>::total;
        case 2561: return Geo<256, 1>::total; case 2562: return Geo<256, 2>::total; case 2564: return Geo<256, 4>::total;
        default: return 0;
    }
}
