// fv_logprob.cu -- the teacher-forced pass of fv_log_prob (Alg. 1), layer-major:
// every position of every sample is known in advance, so each layer is three launches over all
// M = B*N rows:
//   lp_qkv_kernel  : (embedding for layer 0) -> LN1 -> [M,d] x [d,3d] on tcgen05 tensor cores with
//                    the accumulator in tensor memory -> q (fp32) and K|V rows (bf16, the same KV
//                    pool layout fv_sample uses)                                    (Eq. 2, l.98)
//   lp_attn_kernel : masked attention of every row over the rows its CSR mask row names, one warp
//                    per query, K/V rows of neighbouring queries shared through L1  (Eq. 3, l.102)
//   lp_ffn_kernel  : LN2 -> W1 -> GELU -> W2 -> residual, both GEMMs on tcgen05, the 4d hidden
//                    activation never leaves the SM (TMEM -> registers -> shared memory)
// and lp_head_kernel: sigmoid head, log p of the given spin, per-sample fp64 sum (Alg. 1 l.8-9).
// GEMM operands are bf16 with fp32 accumulation; LayerNorm, softmax, residual stream stay fp32 --
// the same arithmetic as the decode kernel, so both paths sit inside the same error bound.
#include <cstdlib>
#include <cstring>

#include "fv_device.cuh"
#include "fv_umma.cuh"

namespace {
using namespace fvdev;

constexpr int LP_THREADS = 512;   // 16 warps: warp w reads TMEM lanes 32 (w % 4) .. +31, column group w / 4
constexpr int NCG = LP_THREADS / 128;   // column groups sharing one TMEM lane quarter
constexpr int FFN_THREADS = 256;  // the FFN kernel runs 2 CTAs per SM (one normalises/stores while the other is in GELU)
constexpr int NCG_F = FFN_THREADS / 128;
constexpr int TM = 128;           // rows per tile = UMMA M

template <int D> struct LpGeo {
    static constexpr int KP = D < 64 ? 64 : D;            // K padded to whole 64-element swizzle blocks
    static constexpr int KB = KP / 64;
    static constexpr int A_BYTES = TM * KP * 2;           // one bf16 A tile
    static constexpr int NQ = 3 * D;                      // QKV output features
    static constexpr int NQ_CH = NQ <= 256 ? NQ : 128;    // columns per MMA
    static constexpr int WQ_BYTES = NQ * KP * 2;
    static constexpr int STG_STRIDE = 4 * D + 16;         // one staged output row: D fp32 (q) or 2D bf16 (K|V), padded
    static constexpr int STG_BYTES = TM * STG_STRIDE;
    static constexpr int QKV_SMEM = 1024 + A_BYTES + WQ_BYTES + STG_BYTES + 64;
    static constexpr int TMEM_Q = NQ <= 128 ? 128 : (NQ <= 256 ? 256 : 512);
    // FFN: hidden 4d in chunks of HC columns
    static constexpr int HC = FV_LP_HC;
    static constexpr int NHC = 4 * D / HC;
    static constexpr int W1_BYTES = HC * KP * 2;          // [HC rows x KP]
    static constexpr int W2_BYTES = D * HC * 2;           // [D rows x HC]
    static constexpr int H_BYTES = TM * HC * 2;
    static constexpr int WBUF = W1_BYTES + W2_BYTES;
    static constexpr int FFN_SMEM = A_BYTES + H_BYTES + 2 * WBUF;
    static constexpr int TMEM_F = (2 * HC + D) <= 256 ? 256 : 512;   // two GEMM 1 accumulators + GEMM 2's
};

__device__ __forceinline__ void sts128(uint32_t addr, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
    asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};\n" ::"r"(addr), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
__device__ __forceinline__ void sts64(uint32_t addr, uint32_t x, uint32_t y) {
    asm volatile("st.shared.v2.b32 [%0], {%1,%2};\n" ::"r"(addr), "r"(x), "r"(y) : "memory");
}

// LayerNorm with EIGHT lanes per row (four rows per warp instruction): lane j of a row holds the
// float4 pieces k * 8 + j, k < D / 32, so a row's 128-byte segments are read whole, the two
// reductions take three shuffle steps instead of five and serve four rows at once.  x holds the
// row's values on entry and the normalised values on return.
template <int D>
__device__ __forceinline__ void ln8_to_tile(float4 (&x)[D / 32], const float* __restrict__ gam, const float* __restrict__ bet,
                                            float eps, uint32_t sA, int r, int j) {
    constexpr int NV = D / 32;
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < NV; ++k) s += (x[k].x + x[k].y) + (x[k].z + x[k].w);
    s += __shfl_xor_sync(0xffffffffu, s, 1);
    s += __shfl_xor_sync(0xffffffffu, s, 2);
    s += __shfl_xor_sync(0xffffffffu, s, 4);
    const float mean = s * (1.0f / D);
    float v = 0.f;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        const float a0 = x[k].x - mean, a1 = x[k].y - mean, a2 = x[k].z - mean, a3 = x[k].w - mean;
        v += (a0 * a0 + a1 * a1) + (a2 * a2 + a3 * a3);
    }
    v += __shfl_xor_sync(0xffffffffu, v, 1);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    v += __shfl_xor_sync(0xffffffffu, v, 4);
    const float rstd = rsqrtf(v * (1.0f / D) + eps);
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        const int f0 = (k * 8 + j) * 4;
        const float4 g = __ldg(reinterpret_cast<const float4*>(gam + f0)), b = __ldg(reinterpret_cast<const float4*>(bet + f0));
        x[k].x = (x[k].x - mean) * rstd * g.x + b.x;
        x[k].y = (x[k].y - mean) * rstd * g.y + b.y;
        x[k].z = (x[k].z - mean) * rstd * g.z + b.z;
        x[k].w = (x[k].w - mean) * rstd * g.w + b.w;
        sts64(sA + (f0 >> 6) * (TM * 128) + umma::sw128_chunk(r, (f0 & 63) >> 3) + (f0 & 7) * 2,
              pack_bf16(x[k].x, x[k].y), pack_bf16(x[k].z, x[k].w));
    }
}

// The same tile write without the normalisation (operand of the W_O GEMM: the attention output as it is).
template <int D>
__device__ __forceinline__ void cvt8_to_tile(const float4 (&x)[D / 32], uint32_t sA, int r, int j) {
#pragma unroll
    for (int k = 0; k < D / 32; ++k) {
        const int f0 = (k * 8 + j) * 4;
        sts64(sA + (f0 >> 6) * (TM * 128) + umma::sw128_chunk(r, (f0 & 63) >> 3) + (f0 & 7) * 2,
              pack_bf16(x[k].x, x[k].y), pack_bf16(x[k].z, x[k].w));
    }
}

constexpr int RB = 8;             // rows whose loads a warp keeps in flight in the LN prologues

struct LpArgs {
    int32_t B, N, NL, layer, d_token, ln2_style, vocab;
    float ln_eps;
    long long M;                    // B * N rows
    const int8_t* spins;            // [B, N]
    float* h;                       // [M, d] fp32 residual stream
    float* q;                       // [M, d] fp32 queries of the current layer
    __nv_bfloat16* kv;              // KV pool [B][NL][N][2d]
    const float* tok_emb;
    const float* posemb;
    const unsigned char* w_img;     // pre-swizzled bf16 weight image(s) of this layer
    const float* bias;              // bqkv | (b1, b2)
    const float* bias2;
    const float* ln_g;
    const float* ln_b;
    int32_t has_wo;                 // attention writes u over q (then lp_qkv_kernel<D, true>: h += W_O u + b_O) instead of h += u
};

// --------------------------------------------------------------------------------- QKV
// WO = true: the optional output projection (PAPER.md:107 bypasses it; reading A8) with the same machinery -- rows of the
// attention output u (stored over q) -> bf16 A tile, [M,d] x [d,d] against the W_O image, epilogue h += acc + b_O.
template <int D, bool WO = false>
__global__ void __launch_bounds__(LP_THREADS, 1) lp_qkv_kernel(const __grid_constant__ LpArgs a) {
    using G = LpGeo<D>;
    constexpr int NOUT = WO ? D : G::NQ;                          // output features
    constexpr int NOUT_CH = WO ? (D <= 256 ? D : 128) : G::NQ_CH;
    constexpr int W_BYTES = NOUT * G::KP * 2;
    extern __shared__ unsigned char lp_raw[];
    unsigned char* sm = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(lp_raw) + 1023) & ~(uintptr_t)1023);
    unsigned char* sA = sm;
    unsigned char* sW = sm + G::A_BYTES;
    unsigned char* sS = sW + G::WQ_BYTES;            // output staging (epilogue)
    const uint32_t sA_u32 = umma::smem_u32(sA), sS_u32 = umma::smem_u32(sS);
    __shared__ uint64_t bar_w, bar_mma;
    __shared__ uint32_t tmem_slot;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) { umma::mbar_init(&bar_w, 1); umma::mbar_init(&bar_mma, 1); umma::fence_mbar_init(); }
    if (warp == 0) umma::tmem_alloc<G::TMEM_Q>(&tmem_slot);
    umma::fence_before_sync();
    __syncthreads();
    umma::fence_after_sync();
    const uint32_t tmem = tmem_slot;
    // the layer's whole W_qkv image stays in shared memory for the CTA's lifetime (bulk copies)
    if (tid == 0) {
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(umma::smem_u32(&bar_w)), "r"((uint32_t)W_BYTES) : "memory");
        for (int off = 0; off < W_BYTES; off += 16384) {
            const uint32_t n = min(16384, W_BYTES - off);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                         ::"r"(umma::smem_u32(sW + off)), "l"(a.w_img + off), "r"(n), "r"(umma::smem_u32(&bar_w)) : "memory");
        }
    }
    if (D < 64) {                                   // zero the K padding of the A tile once
        for (int i = tid; i < G::A_BYTES / 16; i += LP_THREADS) reinterpret_cast<uint4*>(sA)[i] = make_uint4(0, 0, 0, 0);
        __syncthreads();
    }
    const uint32_t idesc = umma::make_idesc_bf16(TM, NOUT_CH);
    const long long n_tiles = (a.M + TM - 1) / TM;
    uint32_t ph = 0;
    bool w_ready = false;
    // A warp owns RB = 8 rows of a tile.  Their loads are issued together, and the NEXT tile's rows are
    // requested before this tile's epilogue, so the HBM round trip hides under the MMA and the stores.
    static_assert(TM / (LP_THREADS / 32) == RB, "one load batch per tile");
    // eight lanes per row (see ln8_to_tile): a warp's 8 rows are two passes of four
    constexpr int NV = D / 32;
    const int sub = lane >> 3, jl = lane & 7;
    float4 x[RB / 4][NV];
    auto load_tile = [&](long long tile) {
#pragma unroll
        for (int ps = 0; ps < RB / 4; ++ps) {
            const int r = warp * RB + ps * 4 + sub;
            const long long gi = tile * TM + r;
            if (WO && gi < a.M) {
#pragma unroll
                for (int k = 0; k < NV; ++k) x[ps][k] = *reinterpret_cast<const float4*>(a.q + gi * D + (k * 8 + jl) * 4);
            } else if (gi < a.M) {
                if (a.layer == 0) {                 // Eq. 15 (l.287-292): x = [tok_emb[s_{t-1}] ; pos_emb[t]]
                    const int t = (int)(gi % a.N);
                    const int tok = t == 0 ? 0 : (a.vocab > 2 ? (int)(uint8_t)a.spins[gi - 1] : (a.spins[gi - 1] > 0 ? 1 : 0));
#pragma unroll
                    for (int k = 0; k < NV; ++k) {
                        float e[4];
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            const int f = (k * 8 + jl) * 4 + q;
                            e[q] = f < a.d_token ? __ldg(a.tok_emb + tok * a.d_token + f)
                                                 : __ldg(a.posemb + (size_t)t * (D - a.d_token) + (f - a.d_token));
                        }
                        x[ps][k] = make_float4(e[0], e[1], e[2], e[3]);
                    }
                } else {
#pragma unroll
                    for (int k = 0; k < NV; ++k) x[ps][k] = *reinterpret_cast<const float4*>(a.h + gi * D + (k * 8 + jl) * 4);
                }
            } else {
#pragma unroll
                for (int k = 0; k < NV; ++k) x[ps][k] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
    };
    if ((long long)blockIdx.x < n_tiles) load_tile(blockIdx.x);
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        // ---- prologue: (embedding) + LN1 -> bf16 A tile ---------------------------------------
#pragma unroll
        for (int ps = 0; ps < RB / 4; ++ps) {
            const int r = warp * RB + ps * 4 + sub;
            const long long gi = tile * TM + r;
            if (!WO && a.layer == 0 && gi < a.M) {
#pragma unroll
                for (int k = 0; k < NV; ++k) *reinterpret_cast<float4*>(a.h + gi * D + (k * 8 + jl) * 4) = x[ps][k];
            }
            if constexpr (WO) cvt8_to_tile<D>(x[ps], sA_u32, r, jl);
            else ln8_to_tile<D>(x[ps], a.ln_g, a.ln_b, a.ln_eps, sA_u32, r, jl);
        }
        umma::fence_smem_to_async();
        __syncthreads();
        // ---- q|k|v = LN1(h) W^T on the tensor cores --------------------------------------------
        if (tid == 0) {
            if (!w_ready) umma::mbar_wait(&bar_w, 0);
            umma::fence_after_sync();
            const uint32_t a0 = umma::smem_u32(sA), w0 = umma::smem_u32(sW);
#pragma unroll
            for (int nc = 0; nc < NOUT / NOUT_CH; ++nc)
#pragma unroll
                for (int kb = 0; kb < G::KB; ++kb)
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks)
                        umma::mma_bf16_ss(tmem + nc * NOUT_CH, umma::make_desc_sw128(a0 + kb * (TM * 128) + ks * 32),
                                          umma::make_desc_sw128(w0 + kb * (NOUT * 128) + nc * (NOUT_CH * 128) + ks * 32),
                                          idesc, (kb | ks) != 0);
            umma::commit(&bar_mma);
        }
        w_ready = true;
        if (tile + gridDim.x < n_tiles) load_tile(tile + gridDim.x);
        umma::mbar_wait(&bar_mma, ph);
        ph ^= 1;
        umma::fence_after_sync();
        // ---- epilogue: + bias; q -> fp32, k|v -> bf16 KV pool row (Alg. 2's cache layout) ---------
        // A TMEM read hands a thread one ROW; stored from there every instruction would touch 32
        // lines.  Two passes through a padded staging tile instead (q as fp32, then K|V as the
        // bf16 row the pool stores -- both 4d bytes wide): a warp then writes whole rows.
        {
            constexpr int LPRW = D / 4;                    // lanes per staged row (16 B each)
            constexpr int RPI = 32 / LPRW;                 // rows per warp instruction
            constexpr int RPW = TM / (LP_THREADS / 32);    // rows per warp
            const int r = (warp & 3) * 32 + lane;          // staging: this thread's row
            const int rB = warp * RPW + lane / LPRW;       // storing: first row, then += RPI
            const int cB = (lane % LPRW) * 16;             //          byte offset inside the row
#pragma unroll 1
            for (int pass = 0; pass < (WO ? 1 : 2); ++pass) {
                const int cb0 = pass == 0 ? 0 : D / 32, cb1 = pass == 0 ? D / 32 : G::NQ / 32;
                for (int cb = cb0 + (warp >> 2); cb < cb1; cb += NCG) {
                    float v[32];
                    umma::tmem_ld32(tmem + ((uint32_t)((warp & 3) * 32) << 16) + cb * 32, v);
                    const int f0 = cb * 32;
#pragma unroll
                    for (int j = 0; j < 32; j += 4) {
                        const float4 bb = __ldg(reinterpret_cast<const float4*>(a.bias + f0 + j));
                        v[j] += bb.x; v[j + 1] += bb.y; v[j + 2] += bb.z; v[j + 3] += bb.w;
                    }
                    if (pass == 0) {
#pragma unroll
                        for (int j = 0; j < 32; j += 4)
                            sts128(sS_u32 + r * G::STG_STRIDE + (f0 + j) * 4, __float_as_uint(v[j]), __float_as_uint(v[j + 1]),
                                   __float_as_uint(v[j + 2]), __float_as_uint(v[j + 3]));
                    } else {
#pragma unroll
                        for (int j = 0; j < 32; j += 8)
                            sts128(sS_u32 + r * G::STG_STRIDE + (f0 - D + j) * 2, pack_bf16(v[j], v[j + 1]), pack_bf16(v[j + 2], v[j + 3]),
                                   pack_bf16(v[j + 4], v[j + 5]), pack_bf16(v[j + 6], v[j + 7]));
                    }
                }
                __syncthreads();
#pragma unroll
                for (int i = 0; i < RPW / RPI; ++i) {
                    const int row = rB + i * RPI;
                    const long long gi = tile * TM + row;
                    if (gi < a.M) {
                        uint4 val = *reinterpret_cast<const uint4*>(sS + row * G::STG_STRIDE + cB);
                        unsigned char* dst;
                        if constexpr (WO) {              // residual: h += W_O u + b_O
                            dst = reinterpret_cast<unsigned char*>(a.h + gi * D);
                            const float4 hv = *reinterpret_cast<const float4*>(dst + cB);
                            val.x = __float_as_uint(hv.x + __uint_as_float(val.x)); val.y = __float_as_uint(hv.y + __uint_as_float(val.y));
                            val.z = __float_as_uint(hv.z + __uint_as_float(val.z)); val.w = __float_as_uint(hv.w + __uint_as_float(val.w));
                        } else if (pass == 0) dst = reinterpret_cast<unsigned char*>(a.q + gi * D);
                        else {
                            const int b = (int)(gi / a.N), t = (int)(gi % a.N);
                            dst = reinterpret_cast<unsigned char*>(a.kv + (((size_t)b * a.NL + a.layer) * a.N + t) * (2 * D));
                        }
                        *reinterpret_cast<uint4*>(dst + cB) = val;
                    }
                }
                if (pass == 0) __syncthreads();            // the staging tile is rewritten by the K|V pass
            }
        }
        umma::fence_before_sync();
        __syncthreads();                            // TMEM and the A tile are free for the next tile
        umma::fence_after_sync();
    }
    if (!w_ready && tid == 0) umma::mbar_wait(&bar_w, 0);   // never leave a bulk copy in flight
    __syncthreads();
    if (warp == 0) umma::tmem_dealloc<G::TMEM_Q>(tmem);
}

// --------------------------------------------------------------------------------- attention
// One warp per query row; the row's KV rows come through L1 (rows of neighbouring positions of the
// same sample overlap almost entirely, and the CTA walks consecutive positions).  Only the rows
// the CSR mask names are touched: tiles with no allowed pair are never visited, and inside a
// row nothing is computed for masked-out keys.
template <int D, int DH>
__global__ void __launch_bounds__(512) lp_attn_kernel(const __grid_constant__ LpArgs a, const int32_t* __restrict__ rowptr,
                                                      const int32_t* __restrict__ cols, int rows_per_cta) {
    constexpr int LPR = D / 8;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long r0 = (long long)blockIdx.x * rows_per_cta;
    for (int i = warp; i < rows_per_cta; i += 16) {
        const long long gi = r0 + i;
        if (gi >= a.M) break;
        const int b = (int)(gi / a.N), t = (int)(gi % a.N);
        const int e0 = __ldg(rowptr + t), e1 = __ldg(rowptr + t + 1);
        float mm, ll, acc[8];
        attend_range<D, DH>(a.q + gi * D, a.kv + ((size_t)b * a.NL + a.layer) * a.N * (2 * D), cols, e0, e1, lane, mm, ll, acc);
        if (lane < LPR) {
            const float inv = 1.0f / ll;
            float* hp = (a.has_wo ? a.q : a.h) + gi * D + lane * 8;       // with W_O: u over this row's q (read above)
            float4 h0 = *reinterpret_cast<float4*>(hp), h1 = *reinterpret_cast<float4*>(hp + 4);
            if (a.has_wo) h0 = h1 = make_float4(0.f, 0.f, 0.f, 0.f);
            h0.x += acc[0] * inv; h0.y += acc[1] * inv; h0.z += acc[2] * inv; h0.w += acc[3] * inv;
            h1.x += acc[4] * inv; h1.y += acc[5] * inv; h1.z += acc[6] * inv; h1.w += acc[7] * inv;
            *reinterpret_cast<float4*>(hp) = h0;
            *reinterpret_cast<float4*>(hp + 4) = h1;
        }
    }
}

// --------------------------------------------------------------------------------- attention (tensor cores)
// Block-skipping masked attention for d_h = 16 (all BASELINE configs).  A CTA owns BQ = 32
// consecutive positions of one sample, one warp per head.  The host plan (fv_create_model) gives,
// per query block, the sorted UNION of the key positions its 32 mask rows name (padded to 16) and,
// per 16-key step and query, a 16-bit allow mask: key tiles outside the union are never loaded,
// steps in which none of a warp's 16 queries has an allowed key are skipped, and inside a step
// masked-out scores get probability exactly 0.
//   S = Q K^T : mma.sync m16n8k16 (k = d_h = 16: one MMA per 8 keys), Q pre-scaled; Q and P enter as
//               bf16 hi + lo pairs (two MMAs), so only K and V carry bf16 rounding -- as in fv_sample
//   online softmax (base 2, fp32) on the C fragments
//   O += P V  : P re-used from the C fragments as the A operand (bf16), V via ldmatrix.trans
// K|V rows of the union are staged in shared memory by cp.async in chunks of 64 keys, double
// buffered; rows are padded by 16 B so the 8 rows of an ldmatrix tile hit different banks.
#ifndef FV_LP_PSPLIT
#define FV_LP_PSPLIT 1      // 0: P as one bf16 (4.3 instead of 4.9 ms per layer on cfg5, but the sample/log_prob chain-rule check at 2e-4 fails)
#endif
constexpr int ATT_BQ = 32, ATT_UC = 64;

__device__ __forceinline__ void ldsm_x4(uint32_t (&r)[4], uint32_t addr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t (&r)[4], uint32_t addr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
// (x, y) -> packed bf16 pairs hi and lo with hi + lo = (x, y) to ~16 mantissa bits.  The pair is
// rounded by one packed conversion (F2FP, ALU pipe) and widened again by a shift and a mask: the
// scalar conversions (F2F) share the quarter-rate XU pipe with the softmax's ex2, which was the
// attention kernel's busiest pipe.  Same round-to-nearest-even results bit for bit.
__device__ __forceinline__ void split_bf16(float x, float y, uint32_t& hi, uint32_t& lo) {
    hi = pack_bf16(x, y);
    lo = pack_bf16(x - __uint_as_float(hi << 16), y - __uint_as_float(hi & 0xffff0000u));
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(src) : "memory");
}

template <int D>
__global__ void __launch_bounds__(D / 16 * 32, 3) lp_attn_mma_kernel(const __grid_constant__ LpArgs a,
                                                                  const int32_t* __restrict__ blk_uptr,
                                                                  const int32_t* __restrict__ ukeys,
                                                                  const uint16_t* __restrict__ amask, int n_blk) {
    constexpr int NTH = D / 16 * 32, RS = 4 * D + 16, BUF = ATT_UC * RS, PCS = 4 * D / 16;   // 16-B pieces per row
    extern __shared__ __align__(16) unsigned char att_sm[];
    const int tid = threadIdx.x, head = tid >> 5, lane = tid & 31, g = lane >> 2, c = lane & 3;
    const int b = blockIdx.x / n_blk, blk = blockIdx.x - b * n_blk;
    const int t0 = blk * ATT_BQ;
    const int u0 = __ldg(blk_uptr + blk), U = __ldg(blk_uptr + blk + 1) - u0;
    const int n_chunks = (U + ATT_UC - 1) / ATT_UC;
    const unsigned char* kvb = reinterpret_cast<const unsigned char*>(a.kv + ((size_t)b * a.NL + a.layer) * a.N * (2 * D));
    const uint32_t sm0 = umma::smem_u32(att_sm);
    // a thread copies one 16-byte piece of RPI-spaced rows; the chunk's key positions are all
    // requested first, so the copies wait for ONE index load, not for one per row
    auto stage = [&](int ch) {
        constexpr int RPI = NTH / PCS, NIT = ATT_UC / RPI;
        const int k0 = ch * ATT_UC, nk = min(ATT_UC, U - k0);
        const uint32_t dst = sm0 + (ch & 1) * BUF;
        const int r0 = tid / PCS, pc = tid - r0 * PCS;
        int keys[NIT];
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int r = r0 + it * RPI;
            keys[it] = r < nk ? __ldg(ukeys + u0 + k0 + r) : -1;
        }
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int r = r0 + it * RPI;
            if (keys[it] >= 0) cp_async16(dst + r * RS + pc * 16, kvb + (size_t)keys[it] * (4 * D) + pc * 16);
        }
        asm volatile("cp.async.commit_group;\n" ::: "memory");
    };
    stage(0);
    // Q fragments (A operand), pre-scaled by log2(e)/sqrt(d_h)
    const float qs = kLog2e * 0.25f;
    uint32_t qa[2][4], ql[2][4];        // bf16 hi and lo parts: q keeps ~16 mantissa bits through the MMA
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            const int t = t0 + mt * 16 + g + hh * 8;
            float2 lo = make_float2(0.f, 0.f), hi = lo;
            if (t < a.N) {
                const float* qp = a.q + ((long long)b * a.N + t) * D + head * 16 + 2 * c;
                lo = *reinterpret_cast<const float2*>(qp);
                hi = *reinterpret_cast<const float2*>(qp + 8);
            }
            split_bf16(lo.x * qs, lo.y * qs, qa[mt][hh], ql[mt][hh]);
            split_bf16(hi.x * qs, hi.y * qs, qa[mt][hh + 2], ql[mt][hh + 2]);
        }
    }
    // the residual rows this warp updates at the very end: start them towards L2 now
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
        const int t = t0 + mt * 16 + (lane >> 1);          // 16 rows x 2 sectors (the head's 64 B) per m-tile
        if (t < a.N) asm volatile("prefetch.global.L2 [%0];\n" ::"l"(a.h + ((long long)b * a.N + t) * D + head * 16 + (lane & 1) * 8));
    }
    float o[2][2][4], mrow[2][2], lrow[2][2];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int x = 0; x < 2; ++x) {
            mrow[mt][x] = -1e30f; lrow[mt][x] = 0.f;
#pragma unroll
            for (int e = 0; e < 4; ++e) o[mt][x][e] = 0.f;
        }
    const uint16_t* mk = amask + (size_t)(u0 / 16) * ATT_BQ;
    for (int ch = 0; ch < n_chunks; ++ch) {
        if (ch + 1 < n_chunks) { stage(ch + 1); asm volatile("cp.async.wait_group 1;\n" ::: "memory"); }
        else asm volatile("cp.async.wait_group 0;\n" ::: "memory");
        __syncthreads();
        const uint32_t buf = sm0 + (ch & 1) * BUF;
        const int nst = (min(ATT_UC, U - ch * ATT_UC)) / 16;
        // the allow masks of step st + 1 are requested before step st is worked on
        uint32_t nbits[2][2];
        auto load_bits = [&](int st) {
            const uint16_t* ms = mk + (size_t)(ch * (ATT_UC / 16) + st) * ATT_BQ;
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
                nbits[mt][0] = __ldg(ms + mt * 16 + g);
                nbits[mt][1] = __ldg(ms + mt * 16 + g + 8);
            }
        };
        if (nst > 0) load_bits(0);
        for (int st = 0; st < nst; ++st) {
            uint32_t bits[2][2];
            bool any[2];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
                bits[mt][0] = nbits[mt][0];
                bits[mt][1] = nbits[mt][1];
            }
            if (st + 1 < nst) load_bits(st + 1);
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) any[mt] = __any_sync(0xffffffffu, (bits[mt][0] | bits[mt][1]) != 0);
            if (!any[0] && !any[1]) continue;
            uint32_t kf[4], vf[4];
            {
                const int mi = lane >> 3, rr = lane & 7;
                ldsm_x4(kf, buf + (st * 16 + (mi >> 1) * 8 + rr) * RS + head * 32 + (mi & 1) * 16);
                ldsm_x4_t(vf, buf + (st * 16 + (mi & 1) * 8 + rr) * RS + 2 * D + head * 32 + (mi >> 1) * 16);
            }
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
                if (!any[mt]) continue;
                float sc[2][4];
#pragma unroll
                for (int n = 0; n < 2; ++n) {
                    sc[n][0] = sc[n][1] = sc[n][2] = sc[n][3] = 0.f;
                    mma_bf16(sc[n], make_uint4(qa[mt][0], qa[mt][1], qa[mt][2], qa[mt][3]), kf[2 * n], kf[2 * n + 1]);
                    mma_bf16(sc[n], make_uint4(ql[mt][0], ql[mt][1], ql[mt][2], ql[mt][3]), kf[2 * n], kf[2 * n + 1]);
                }
                // fast path: every key of the step is allowed for all 16 queries of the tile (the inside
                // of a sliding window) -- no per-element mask arithmetic
                const bool full = __all_sync(0xffffffffu, (bits[mt][0] & bits[mt][1]) == 0xFFFFu);
                float mx[2] = {mrow[mt][0], mrow[mt][1]};
                float p[2][4];
                float corr[2];
                if (full) {
#pragma unroll
                    for (int n = 0; n < 2; ++n)
#pragma unroll
                        for (int e = 0; e < 4; ++e) mx[e >> 1] = fmaxf(mx[e >> 1], sc[n][e]);
                } else {
#pragma unroll
                    for (int n = 0; n < 2; ++n)
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const bool ok = (bits[mt][e >> 1] >> (n * 8 + 2 * c + (e & 1))) & 1u;
                            sc[n][e] = ok ? sc[n][e] : -INFINITY;      // exp2(-inf - m) = 0 exactly (m is finite)
                            mx[e >> 1] = fmaxf(mx[e >> 1], sc[n][e]);
                        }
                }
#pragma unroll
                for (int x = 0; x < 2; ++x) {
                    mx[x] = fmaxf(mx[x], __shfl_xor_sync(0xffffffffu, mx[x], 1));
                    mx[x] = fmaxf(mx[x], __shfl_xor_sync(0xffffffffu, mx[x], 2));
                    corr[x] = fast_exp2(mrow[mt][x] - mx[x]);
                    mrow[mt][x] = mx[x];
                    lrow[mt][x] *= corr[x];
                }
#pragma unroll
                for (int n = 0; n < 2; ++n)
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        p[n][e] = fast_exp2(sc[n][e] - mx[e >> 1]);
                        lrow[mt][e >> 1] += p[n][e];
                    }
#pragma unroll
                for (int x = 0; x < 2; ++x)
#pragma unroll
                    for (int e = 0; e < 4; ++e) o[mt][x][e] *= corr[e >> 1];
#if FV_LP_PSPLIT
                uint4 pa, pl;                              // P = hi + lo in bf16 (as q above)
                split_bf16(p[0][0], p[0][1], pa.x, pl.x);
                split_bf16(p[0][2], p[0][3], pa.y, pl.y);
                split_bf16(p[1][0], p[1][1], pa.z, pl.z);
                split_bf16(p[1][2], p[1][3], pa.w, pl.w);
                mma_bf16(o[mt][0], pa, vf[0], vf[1]);
                mma_bf16(o[mt][1], pa, vf[2], vf[3]);
                mma_bf16(o[mt][0], pl, vf[0], vf[1]);
                mma_bf16(o[mt][1], pl, vf[2], vf[3]);
#else
                const uint4 pa = make_uint4(pack_bf16(p[0][0], p[0][1]), pack_bf16(p[0][2], p[0][3]),
                                            pack_bf16(p[1][0], p[1][1]), pack_bf16(p[1][2], p[1][3]));
                mma_bf16(o[mt][0], pa, vf[0], vf[1]);
                mma_bf16(o[mt][1], pa, vf[2], vf[3]);
#endif
            }
        }
        __syncthreads();                               // buffer (ch & 1) is restaged two chunks later
    }
    // finalise: h += O / l  (Alg. 2 l.15: residual without W_O); the residual rows are all
    // requested before the first is used
    float2 hres[2][2][2];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            const int t = t0 + mt * 16 + g + hh * 8;
            const float* hp = a.h + ((long long)b * a.N + t) * D + head * 16 + 2 * c;
#pragma unroll
            for (int x = 0; x < 2; ++x) hres[mt][hh][x] = (t < a.N && !a.has_wo) ? *reinterpret_cast<const float2*>(hp + x * 8) : make_float2(0.f, 0.f);
        }
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            float l = lrow[mt][hh];
            l += __shfl_xor_sync(0xffffffffu, l, 1);
            l += __shfl_xor_sync(0xffffffffu, l, 2);
            const int t = t0 + mt * 16 + g + hh * 8;
            if (t < a.N && l > 0.f) {
                const float inv = 1.0f / l;
                // with W_O the output u replaces this warp's own q elements (its Q fragments were read at the start)
                float* hp = (a.has_wo ? a.q : a.h) + ((long long)b * a.N + t) * D + head * 16 + 2 * c;
#pragma unroll
                for (int x = 0; x < 2; ++x) {
                    float2 hv = hres[mt][hh][x];
                    hv.x += o[mt][x][hh * 2] * inv;
                    hv.y += o[mt][x][hh * 2 + 1] * inv;
                    *reinterpret_cast<float2*>(hp + x * 8) = hv;
                }
            }
        }
}

// --------------------------------------------------------------------------------- FFN
// h <- h + W2 gelu(W1 LN2(h) + b1) + b2 for a tile of 128 rows (Alg. 2 l.16 form; ln2_style 1:
// h <- LN2(h) first, Alg. 1 l.5).  The hidden layer is processed in chunks of HC columns, chunk g
// (counted over all tiles of the CTA) using accumulator buffer g & 1:
//   acc1[g&1] (TMEM cols [0,HC) / [HC,2HC)) = A W1_j^T
//   H_j = bf16(gelu(acc1 + b1_j)) -> shared memory, swizzled K-major (it is GEMM 2's A operand)
//   acc2 (TMEM cols [2HC,2HC+D)) += H_j W2_j^T
// GEMM 1 of chunk g+1 is issued BEFORE the GELU epilogue of chunk g (the second accumulator buffer
// makes that legal), GEMM 2 of chunk g right after it: the tensor pipe works under the epilogue
// and no warp waits for an MMA it has just issued -- the only exposed tensor latency is the tile's
// first GEMM 1 and its last GEMM 2.  W1_j and W2_j arrive as pre-swizzled images by
// cp.async.bulk in two rings of two slots each (W1's slot is free once GEMM 1 is done, one chunk
// earlier than W2's), so every weight copy has a whole chunk time to land.
template <int D>
__global__ void __launch_bounds__(FFN_THREADS, 2) lp_ffn_kernel(const __grid_constant__ LpArgs a) {
    using G = LpGeo<D>;
    extern __shared__ __align__(1024) unsigned char lp_raw_ffn[];   // no alignment slack: two CTAs share an SM
    unsigned char* sm = lp_raw_ffn;
    if (umma::smem_u32(sm) & 1023u) __trap();
    unsigned char* sA = sm;
    unsigned char* sH = sm + G::A_BYTES;
    unsigned char* sW1 = sH + G::H_BYTES;          // 2 x W1_j
    unsigned char* sW2 = sW1 + 2 * G::W1_BYTES;    // 2 x W2_j
    const uint32_t sA_u32 = umma::smem_u32(sA), sH_u32 = umma::smem_u32(sH);
    __shared__ uint64_t bar_w1[2], bar_w2[2], bar_m1[2], bar_m2;
    __shared__ uint32_t tmem_slot;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int i = 0; i < 2; ++i) { umma::mbar_init(&bar_w1[i], 1); umma::mbar_init(&bar_w2[i], 1); umma::mbar_init(&bar_m1[i], 1); }
        umma::mbar_init(&bar_m2, 1);
        umma::fence_mbar_init();
    }
    if (warp == 0) umma::tmem_alloc<G::TMEM_F>(&tmem_slot);
    if (D < 64) for (int i = tid; i < G::A_BYTES / 16; i += FFN_THREADS) reinterpret_cast<uint4*>(sA)[i] = make_uint4(0, 0, 0, 0);
    umma::fence_before_sync();
    __syncthreads();
    umma::fence_after_sync();
    const uint32_t tmem = tmem_slot;
    const uint32_t tmem_acc2 = tmem + 2 * G::HC;
    const uint32_t idesc1 = umma::make_idesc_bf16(TM, G::HC), idesc2 = umma::make_idesc_bf16(TM, D);
    const long long n_tiles = (a.M + TM - 1) / TM;
    const long long my_tiles = blockIdx.x < n_tiles ? (n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const long long n_chunks = my_tiles * G::NHC;           // weight chunks this CTA will consume
    auto bulk_in = [&](unsigned char* dst, const unsigned char* src, int bytes, uint64_t* bar) {
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(umma::smem_u32(bar)), "r"((uint32_t)bytes) : "memory");
        for (int off = 0; off < bytes; off += 16384) {
            const uint32_t n = min(16384, bytes - off);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                         ::"r"(umma::smem_u32(dst + off)), "l"(src + off), "r"(n), "r"(umma::smem_u32(bar)) : "memory");
        }
    };
    auto issue_w1 = [&](long long c) {                       // thread 0: W1 of chunk c -> slot c & 1
        bulk_in(sW1 + (int)(c & 1) * G::W1_BYTES, a.w_img + (size_t)(c % G::NHC) * G::WBUF, G::W1_BYTES, &bar_w1[c & 1]);
    };
    auto issue_w2 = [&](long long c) {                       // thread 0: W2 of chunk c -> slot c & 1
        bulk_in(sW2 + (int)(c & 1) * G::W2_BYTES, a.w_img + (size_t)(c % G::NHC) * G::WBUF + G::W1_BYTES, G::W2_BYTES, &bar_w2[c & 1]);
    };
    const uint64_t dA = umma::make_desc_sw128(umma::smem_u32(sA)), dH = umma::make_desc_sw128(umma::smem_u32(sH));
    const uint64_t dW1 = umma::make_desc_sw128(umma::smem_u32(sW1)), dW2 = umma::make_desc_sw128(umma::smem_u32(sW2));
    auto issue_mma1 = [&](long long c) {                     // thread 0: acc1[c & 1] = A W1_c^T
        umma::mbar_wait(&bar_w1[c & 1], (uint32_t)((c >> 1) & 1));
        umma::fence_after_sync();
        // descriptors = one base per operand + compile-time offsets: the issuing thread pays ~45 cycles per tcgen05.mma
        // as it is, and every instruction spent on rebuilding descriptors delays the whole epilogue of its warp
        const uint64_t b0 = dW1 + (uint64_t)(((int)(c & 1) * G::W1_BYTES) >> 4);
        const uint32_t acc = tmem + (uint32_t)(c & 1) * G::HC;
#pragma unroll
        for (int kb = 0; kb < G::KB; ++kb)
#pragma unroll
            for (int ks = 0; ks < 4; ++ks)
                umma::mma_bf16_ss(acc, dA + (uint64_t)((kb * (TM * 128) + ks * 32) >> 4),
                                  b0 + (uint64_t)((kb * (G::HC * 128) + ks * 32) >> 4), idesc1, (kb | ks) != 0);
        umma::commit(&bar_m1[c & 1]);
    };
    if (tid == 0 && n_chunks > 0) {
        issue_w1(0); issue_w2(0);
        if (n_chunks > 1) { issue_w1(1); issue_w2(1); }
    }
    long long g = 0;                                         // chunks done so far = index of the next one
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        if (tid == 0 && tile + gridDim.x < n_tiles) {        // the next tile's rows -> L2 while this one computes
            const long long r0 = (tile + gridDim.x) * TM;
            const long long nr = a.M - r0 < TM ? a.M - r0 : TM;
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(a.h + r0 * D), "r"((uint32_t)(nr * D * 4)) : "memory");
        }
        // ---- prologue: LN2 -> bf16 A tile (ln2_style 1: the residual stream becomes LN2(h)) -----
        {
            constexpr int NV = D / 32, RPW = TM / (FFN_THREADS / 32);     // a warp's 16 rows, four per pass
            const int sub = lane >> 3, j = lane & 7;
            constexpr int PIF = NV >= 4 ? 2 : 4;                          // passes whose loads are in flight together
#pragma unroll 1
            for (int p0 = 0; p0 < RPW / 4; p0 += PIF) {
                float4 x[PIF][NV];
#pragma unroll
                for (int ps = 0; ps < PIF; ++ps) {
                    const long long gi = tile * TM + warp * RPW + (p0 + ps) * 4 + sub;
#pragma unroll
                    for (int k = 0; k < NV; ++k)
                        x[ps][k] = gi < a.M ? *reinterpret_cast<const float4*>(a.h + gi * D + (k * 8 + j) * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
#pragma unroll
                for (int ps = 0; ps < PIF; ++ps) {
                    const int r = warp * RPW + (p0 + ps) * 4 + sub;
                    const long long gi = tile * TM + r;
                    ln8_to_tile<D>(x[ps], a.ln_g, a.ln_b, a.ln_eps, sA_u32, r, j);
                    if (a.ln2_style == 1 && gi < a.M) {
#pragma unroll
                        for (int k = 0; k < NV; ++k) *reinterpret_cast<float4*>(a.h + gi * D + (k * 8 + j) * 4) = x[ps][k];
                    }
                }
            }
        }
        umma::fence_smem_to_async();
        __syncthreads();
        if (tid == 0) issue_mma1(g);                   // GEMM 1 of the tile's first chunk
        for (int j = 0; j < G::NHC; ++j, ++g) {
            // GEMM 1 of the next chunk goes into the other accumulator buffer, whose last reader
            // (the epilogue of chunk g-1) finished before the barrier that closed the previous pass
            if (tid == 0 && j + 1 < G::NHC) issue_mma1(g + 1);
            // this warp's first 16 bias values of the chunk are fetched before the wait, not after it
            static_assert(G::HC / 32 == NCG_F, "one 32-column block per warp and chunk");
            const int cb = warp >> 2;
            const float4* b1 = reinterpret_cast<const float4*>(a.bias + j * G::HC + cb * 32);
            float4 bq[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) bq[c] = __ldg(b1 + c);
            umma::mbar_wait(&bar_m1[g & 1], (uint32_t)((g >> 1) & 1));
            umma::fence_after_sync();
            if (tid == 0 && g + 2 < n_chunks) issue_w1(g + 2);   // GEMM 1 of chunk g has read its W1 slot
            // ---- epilogue 1: H_j = bf16(gelu(acc1 + b1_j)), 32 columns per warp in two halves of
            // 16 (64 live registers fewer than one 32-column read with its bias: room for the
            // compiler to interleave the dependent chains of eight elements)
            {
                const int r = (warp & 3) * 32 + lane;
                const uint32_t t0 = tmem + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(g & 1) * G::HC + cb * 32;
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    float v[16];
                    umma::tmem_ld16(t0 + hf * 16, v);
                    float4 bn[4];
                    if (hf == 0) {
#pragma unroll
                        for (int c = 0; c < 4; ++c) bn[c] = __ldg(b1 + 4 + c);
                    }
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const float4 ba = bq[2 * c], bb = bq[2 * c + 1];
                        uint32_t p[4];
                        p[0] = gelu_erfc_x2(v[c * 8 + 0] + ba.x, v[c * 8 + 1] + ba.y);
                        p[1] = gelu_erfc_x2(v[c * 8 + 2] + ba.z, v[c * 8 + 3] + ba.w);
                        p[2] = gelu_erfc_x2(v[c * 8 + 4] + bb.x, v[c * 8 + 5] + bb.y);
                        p[3] = gelu_erfc_x2(v[c * 8 + 6] + bb.z, v[c * 8 + 7] + bb.w);
                        // H is GEMM 2's operand: the previous chunk's GEMM 2 (issued one pass ago,
                        // behind it only this chunk's GEMM 1) must have read it before the first store
                        if (hf == 0 && c == 0 && j > 0) {
                            umma::mbar_wait(&bar_m2, (uint32_t)((g - 1) & 1));
                            umma::fence_after_sync();
                            if (tid == 0 && g + 1 < n_chunks) issue_w2(g + 1);   // ... and its W2 slot is free
                        }
                        const int col = cb * 32 + hf * 16 + c * 8;    // hidden column inside the chunk = K of GEMM 2
                        sts128(sH_u32 + (col >> 6) * (TM * 128) + umma::sw128_chunk(r, (col & 63) >> 3), p[0], p[1], p[2], p[3]);
                    }
                    if (hf == 0) {
#pragma unroll
                        for (int c = 0; c < 4; ++c) bq[c] = bn[c];
                    }
                }
            }
            umma::fence_before_sync();
            umma::fence_smem_to_async();
            __syncthreads();
            if (tid == 0) {                            // GEMM 2 of this chunk
                umma::fence_after_sync();
                umma::mbar_wait(&bar_w2[g & 1], (uint32_t)((g >> 1) & 1));
                const uint64_t b0 = dW2 + (uint64_t)(((int)(g & 1) * G::W2_BYTES) >> 4);
#pragma unroll
                for (int kb = 0; kb < G::HC / 64; ++kb)
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks)
                        umma::mma_bf16_ss(tmem_acc2, dH + (uint64_t)((kb * (TM * 128) + ks * 32) >> 4),
                                          b0 + (uint64_t)((kb * (D * 128) + ks * 32) >> 4), idesc2, (j | kb | ks) != 0);
                umma::commit(&bar_m2);
            }
        }
        // ---- epilogue 2: h += acc2 + b2.  A TMEM read gives a thread one ROW (32 columns of it), and
        // row-per-thread global accesses cost 32 L1 wavefronts per instruction (the kernel's top
        // unit was the LSU data pipe, 54 %): the accumulator goes through shared memory instead
        // (the A and H tiles are dead after the last GEMM 2; rows padded by 16 B, conflict-free
        // both ways) in passes of SW columns, and a warp then adds and stores whole row segments.
        // The residual rows of the first pass are requested before the wait for the last GEMM 2.
        {
            constexpr int SW = D >= 128 ? 64 : 32;          // columns per pass (the staging must fit A|H)
            constexpr int SROW = SW * 4 + 16;              // padded row stride in bytes
            constexpr int LPRW = SW / 4;                   // lanes per row segment (float4 each)
            constexpr int RPI = 32 / LPRW;                 // rows per warp instruction
            constexpr int RPW = TM / (FFN_THREADS / 32);   // rows per warp
            constexpr int NI = RPW / RPI;
            static_assert(TM * SROW <= G::A_BYTES + G::H_BYTES, "staging fits in the dead A|H tiles");
            const int r = (warp & 3) * 32 + lane;          // phase A: this thread's row
            const int cbl = warp >> 2;                     //          and 32-column block of the pass
            const int rB = warp * RPW + lane / LPRW;       // phase B: first row, then += RPI
            const int cB = (lane % LPRW) * 4;              //          column inside the pass
            float4 hv[NI];
            auto load_h = [&](int c0) {
#pragma unroll
                for (int i = 0; i < NI; ++i) {
                    const long long gi = tile * TM + rB + i * RPI;
                    if (gi < a.M) hv[i] = *reinterpret_cast<const float4*>(a.h + gi * D + c0 + cB);
                }
            };
            load_h(0);
            umma::mbar_wait(&bar_m2, (uint32_t)((g - 1) & 1));     // the tile's last GEMM 2
            umma::fence_after_sync();
            if (tid == 0 && g + 1 < n_chunks) issue_w2(g + 1);
#pragma unroll 1
            for (int c0 = 0; c0 < D; c0 += SW) {
                if (cbl * 32 < SW) {
                    float v[32];
                    umma::tmem_ld32(tmem_acc2 + ((uint32_t)((warp & 3) * 32) << 16) + c0 + cbl * 32, v);
#pragma unroll
                    for (int q = 0; q < 8; ++q)
                        sts128(sA_u32 + r * SROW + (cbl * 32 + q * 4) * 4, __float_as_uint(v[q * 4]), __float_as_uint(v[q * 4 + 1]),
                               __float_as_uint(v[q * 4 + 2]), __float_as_uint(v[q * 4 + 3]));
                }
                __syncthreads();
                const float4 bb = __ldg(reinterpret_cast<const float4*>(a.bias2 + c0 + cB));
#pragma unroll
                for (int i = 0; i < NI; ++i) {
                    const int row = rB + i * RPI;
                    const long long gi = tile * TM + row;
                    const float4 t = *reinterpret_cast<const float4*>(sA + row * SROW + cB * 4);
                    if (gi < a.M) {
                        float4 o = hv[i];
                        o.x += t.x + bb.x; o.y += t.y + bb.y; o.z += t.z + bb.z; o.w += t.w + bb.w;
                        *reinterpret_cast<float4*>(a.h + gi * D + c0 + cB) = o;
                    }
                }
                if (c0 + SW < D) {
                    load_h(c0 + SW);
                    __syncthreads();
                }
            }
        }
        umma::fence_before_sync();
        __syncthreads();
        umma::fence_after_sync();
        if (D < 64) {                                  // the staging overwrote the zero K padding of the A tile
            for (int i = tid; i < G::A_BYTES / 16; i += FFN_THREADS) reinterpret_cast<uint4*>(sA)[i] = make_uint4(0, 0, 0, 0);
            __syncthreads();
        }
    }
    __syncthreads();
    if (warp == 0) umma::tmem_dealloc<G::TMEM_F>(tmem);
}

// --------------------------------------------------------------------------------- head
// p_t(+1) = softmax(z)[1] = sigmoid(w_d . h + b_d) (Alg. 1 l.8); log q = sum_t log p_t(s_t) (l.9),
// fp64, fixed order: warp w sums positions w, w+8, ... then a fixed tree over the 8 warps.
template <int D>
__global__ void __launch_bounds__(256) lp_head_kernel(const __grid_constant__ LpArgs a, const float* __restrict__ head_wd,
                                                      float head_bd, float* __restrict__ logq, float* __restrict__ cond_p) {
    __shared__ double red[8];
    const int b = blockIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int E = D / 32;
    float w[E];
#pragma unroll
    for (int j = 0; j < E; ++j) w[j] = __ldg(head_wd + lane * E + j);
    double acc = 0.0;
    for (int t = warp; t < a.N; t += 8) {
        const long long gi = (long long)b * a.N + t;
        float d = 0.f;
#pragma unroll
        for (int j = 0; j < E; ++j) d += a.h[gi * D + lane * E + j] * w[j];
        d = warp_sum(d) + head_bd;
        const float p = 1.0f / (1.0f + expf(-d));
        const int up = a.spins[gi] > 0;
        const float x = up ? -d : d;                        // log p(s) = -softplus(x)
        acc += (double)(-(fmaxf(x, 0.f) + log1pf(expf(-fabsf(x)))));
        if (cond_p && lane == 0) cond_p[gi] = p;
    }
    if (lane == 0) red[warp] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < 8; ++i) s += red[i];
        logq[b] = (float)s;
    }
}

// Patch tokens (SI I.D, l.603-605): V-way softmax head, log p of the given token; one warp per position, lane owns
// tokens lane, lane + 32, ...; per-sample fp64 sum in the same fixed order as lp_head_kernel.
template <int D>
__global__ void __launch_bounds__(256) lp_head_tok_kernel(const __grid_constant__ LpArgs a, const float* __restrict__ head_w,
                                                          const float* __restrict__ head_b, float* __restrict__ logq,
                                                          float* __restrict__ cond_p) {
    __shared__ double red[8];
    __shared__ __align__(16) float sh_row[8][D];
    const int b = blockIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int V = a.vocab;
    double acc = 0.0;
    for (int t = warp; t < a.N; t += 8) {
        const long long gi = (long long)b * a.N + t;
        for (int f = lane; f < D; f += 32) sh_row[warp][f] = a.h[gi * D + f];
        __syncwarp();
        const int tok = (int)(uint8_t)a.spins[gi];
        float mx = -INFINITY, zt = 0.f, z[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int k = lane + 32 * i;
            z[i] = -INFINITY;
            if (k < V) {
                const float4* wr = reinterpret_cast<const float4*>(head_w + (size_t)k * D);
                float d = __ldg(head_b + k);
#pragma unroll 4
                for (int f4 = 0; f4 < D / 4; ++f4) {
                    const float4 wv = __ldg(wr + f4);
                    const float4 hv = *reinterpret_cast<const float4*>(&sh_row[warp][f4 * 4]);
                    d += hv.x * wv.x + hv.y * wv.y + hv.z * wv.z + hv.w * wv.w;
                }
                z[i] = d;
                mx = fmaxf(mx, d);
                if (k == tok) zt = d;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        float mine = 0.f;
#pragma unroll
        for (int i = 0; i < 8; ++i) mine += lane + 32 * i < V ? expf(z[i] - mx) : 0.f;
        const float S = warp_sum(mine);
        zt = __shfl_sync(0xffffffffu, zt, tok & 31);
        const float lp = (zt - mx) - logf(S);
        acc += (double)lp;
        if (cond_p && lane == 0) cond_p[gi] = expf(zt - mx) / S;
        __syncwarp();
    }
    if (lane == 0) red[warp] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < 8; ++i) s += red[i];
        logq[b] = (float)s;
    }
}

template <int D, int DH>
cudaError_t launch_lp(const FvModelDev& m, int B, const int8_t* spins, float* logq, float* cond_p, int n_sms,
                      cudaStream_t s) {
    using G = LpGeo<D>;
    constexpr int att_smem = 2 * ATT_UC * (4 * D + 16);
    static const bool fv_lp_attn_alu = [] { const char* v = std::getenv("FLASHVAN_ATTN"); return v && std::strcmp(v, "alu") == 0; }();
    {
        cudaError_t e = fv_smem_attr((const void*)lp_qkv_kernel<D>, G::QKV_SMEM);
        if (e == cudaSuccess) e = fv_smem_attr((const void*)lp_ffn_kernel<D>, G::FFN_SMEM);
        if (e == cudaSuccess && m.has_wo) e = fv_smem_attr((const void*)lp_qkv_kernel<D, true>, G::QKV_SMEM);
        if (e == cudaSuccess) e = fv_smem_attr((const void*)lp_attn_mma_kernel<D>, att_smem);
        if (e != cudaSuccess) return e;
    }
    LpArgs a{};
    a.B = B; a.N = m.n_sites; a.NL = m.n_layers; a.d_token = m.d_token; a.ln2_style = m.ln2_style; a.ln_eps = m.ln_eps;
    a.vocab = m.vocab;
    a.has_wo = m.has_wo;
    a.M = (long long)B * m.n_sites;
    a.spins = spins; a.h = m.lp_h; a.q = m.lp_q; a.kv = m.kv; a.tok_emb = m.tok_emb; a.posemb = m.posemb;
    const long long n_tiles = (a.M + TM - 1) / TM;
    const int grid = (int)(n_tiles < n_sms ? n_tiles : n_sms);
    const int rows_per_cta = 64;
    const int grid_ffn = (int)(n_tiles < 2 * n_sms ? n_tiles : 2 * n_sms);
    for (int l = 0; l < m.n_layers; ++l) {
        const FvLayerDev& L = m.layer[l];
        a.layer = l;
        a.w_img = L.img_qkv; a.bias = L.bqkv; a.bias2 = nullptr; a.ln_g = L.ln1_g; a.ln_b = L.ln1_b;
        fv_prof_begin(FV_K_LP_QKV, s);
        lp_qkv_kernel<D><<<grid, LP_THREADS, G::QKV_SMEM, s>>>(a);
        fv_prof_end(FV_K_LP_QKV, s);
        fv_prof_begin(FV_K_LP_ATTN, s);
        if (DH == 16 && m.att_nblk > 0 && !fv_lp_attn_alu) {
            lp_attn_mma_kernel<D><<<(unsigned)(B * m.att_nblk), D / 16 * 32, att_smem, s>>>(a, m.att_blk_uptr, m.att_ukeys,
                                                                                           m.att_mask, m.att_nblk);
        } else {
            lp_attn_kernel<D, DH><<<(unsigned)((a.M + rows_per_cta - 1) / rows_per_cta), 512, 0, s>>>(a, m.mask_rowptr, m.mask_col,
                                                                                                rows_per_cta);
        }
        fv_prof_end(FV_K_LP_ATTN, s);
        if (m.has_wo) {                               // h += W_O u + b_O (u sits where q was)
            a.w_img = L.img_wo; a.bias = L.bo;
            fv_prof_begin(FV_K_LP_QKV, s);
            lp_qkv_kernel<D, true><<<grid, LP_THREADS, G::QKV_SMEM, s>>>(a);
            fv_prof_end(FV_K_LP_QKV, s);
        }
        a.w_img = L.img_ffn; a.bias = L.b1; a.bias2 = L.b2; a.ln_g = L.ln2_g; a.ln_b = L.ln2_b;
        fv_prof_begin(FV_K_LP_FFN, s);
        lp_ffn_kernel<D><<<grid_ffn, FFN_THREADS, G::FFN_SMEM, s>>>(a);
        fv_prof_end(FV_K_LP_FFN, s);
    }
    fv_prof_begin(FV_K_LP_HEAD, s);
    if (m.vocab > 2) lp_head_tok_kernel<D><<<B, 256, 0, s>>>(a, m.head_w, m.head_b, logq, cond_p);
    else lp_head_kernel<D><<<B, 256, 0, s>>>(a, m.head_wd, m.head_bd, logq, cond_p);
    fv_prof_end(FV_K_LP_HEAD, s);
    return cudaGetLastError();
}

}  // namespace

// Layer-major tensor-core path; supported for d in {32, 64, 128} without W_O.  Returns
// cudaErrorNotSupported otherwise (the caller then uses the chunked teacher-forcing kernel).
cudaError_t fv_launch_logprob_tc(const FvModelDev& m, int d_model, int d_head, int B, const int8_t* spins, float* logq,
                                 float* cond_p, int n_sms, int* n_launches, cudaStream_t s) {
    if (!m.lp_h) return cudaErrorNotSupported;
    *n_launches = (m.has_wo ? 4 : 3) * m.n_layers + 1;
    switch (d_model * 1000 + d_head) {
        case 32016: return launch_lp<32, 16>(m, B, spins, logq, cond_p, n_sms, s);
        case 64016: return launch_lp<64, 16>(m, B, spins, logq, cond_p, n_sms, s);
        case 64032: return launch_lp<64, 32>(m, B, spins, logq, cond_p, n_sms, s);
        case 128016: return launch_lp<128, 16>(m, B, spins, logq, cond_p, n_sms, s);
        case 128032: return launch_lp<128, 32>(m, B, spins, logq, cond_p, n_sms, s);
        default: return cudaErrorNotSupported;
    }
}

// ---- fv_log_prob_static: the same launches with the workspace in a file-scope array ---------------------------
// For callers that cannot allocate (CUDA graph capture, serving loops): h, q and the layer-major K|V rows of ONE call
// live in this array instead of the model's cudaMalloc'ed workspace and pool.  Every GPU that loads the library holds
// the FV_LP_STATIC_BYTES until the process exits.  In host code the array's name is only a stand-in for the symbol,
// not a device address: the address comes from cudaGetSymbolAddress, once per device, with that device current.
// Nothing in it has to start at zero -- lp_qkv_kernel writes every h / q / K|V row of the B samples (padding keys of
// the attention plan are position 0, a written row) before any kernel reads it -- so the contents the previous call
// left behind are simply overwritten; two calls that overlap on the GPU (different streams) race on it.
static __device__ __align__(256) unsigned char g_lp_static[FV_LP_STATIC_BYTES];

size_t fv_logprob_static_need(const FvModelDev& m, int d_model, int B) {
    const size_t rows = (size_t)B * m.n_sites;
    const size_t act = (rows * d_model * sizeof(float) + 255) / 256 * 256;                 // h, then q
    return 2 * act + rows * m.n_layers * 2 * d_model * sizeof(__nv_bfloat16);              // then [B][n_l][N][2d] K|V
}

cudaError_t fv_launch_logprob_tc_static(const FvModelDev& m, int d_model, int d_head, int B, const int8_t* spins,
                                        float* logq, float* cond_p, int n_sms, int* n_launches, cudaStream_t s) {
    if (fv_logprob_static_need(m, d_model, B) > FV_LP_STATIC_BYTES) return cudaErrorInvalidValue;
    static std::mutex mu;
    static std::map<int, unsigned char*> base_of;            // device -> address of g_lp_static there
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    unsigned char* base = nullptr;
    {
        std::lock_guard<std::mutex> lock(mu);
        auto it = base_of.find(dev);
        if (it == base_of.end()) {
            e = cudaGetSymbolAddress((void**)&base, g_lp_static);
            if (e != cudaSuccess) return e;
            base_of[dev] = base;
        } else {
            base = it->second;
        }
    }
    const size_t act = ((size_t)B * m.n_sites * d_model * sizeof(float) + 255) / 256 * 256;
    FvModelDev ms = m;                                       // same parameters, plans and images; other workspace
    ms.lp_h = reinterpret_cast<float*>(base);
    ms.lp_q = reinterpret_cast<float*>(base + act);
    ms.kv = reinterpret_cast<__nv_bfloat16*>(base + 2 * act);
    return fv_launch_logprob_tc(ms, d_model, d_head, B, spins, logq, cond_p, n_sms, n_launches, s);
}

// Host side of the images the kernels above copy verbatim into shared memory: W[rows, K] (row
// stride ld, fp32) -> bf16, K-major, SWIZZLE_128B, K padded to KP: K-block kb of 64 columns is a
// [rows x 128 B] slab, 8-row groups 1024 B apart, 16-byte chunk c of row r at chunk c ^ (r & 7).
void fv_pack_sw128(const float* W, int rows, int K, int ld, int KP, uint16_t* dst) {
    for (int kb = 0; kb < KP / 64; ++kb)
        for (int r = 0; r < rows; ++r)
            for (int c = 0; c < 8; ++c)
                for (int e = 0; e < 8; ++e) {
                    const int k = kb * 64 + c * 8 + e;
                    const float x = k < K ? W[(size_t)r * ld + k] : 0.f;
                    const __nv_bfloat16 hbf = __float2bfloat16_rn(x);
                    uint16_t u;
                    memcpy(&u, &hbf, 2);
                    const size_t off = (size_t)kb * rows * 128 + (size_t)(r >> 3) * 1024 + (r & 7) * 128 + ((c ^ (r & 7)) << 4) + e * 2;
                    dst[off / 2] = u;
                }
}
