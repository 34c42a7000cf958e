// fv_device.cuh -- device helpers shared by the forward kernels (fv_forward.cu, fv_decode.cu):
// mma.sync wrapper, packed-weight GEMM over a row tile, LayerNorm row, masked gather attention
// from global memory, shared-memory geometry.
#pragma once
#include "fv_internal.h"

namespace fvdev {


constexpr float kLog2e = 1.4426950408889634f;

__device__ __forceinline__ uint32_t lds32(const void* p) { return *reinterpret_cast<const uint32_t*>(p); }

__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint4& a, uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
        "{%0,%1,%2,%3};\n"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w), "r"(b0), "r"(b1));
}

// Weights are immutable for the kernel's lifetime: read-only path, keep in L1/L2.
__device__ __forceinline__ uint4 ldg_w(const uint4* p) { return __ldg(p); }
// KV rows are written by this CTA earlier in the same kernel: coherent (non-.nc) load.
__device__ __forceinline__ uint4 ld_kv(const void* p) {
    uint4 r;
    asm volatile("ld.global.v4.u32 {%0,%1,%2,%3}, [%4];\n" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

__device__ __forceinline__ float bf_lo(uint32_t x) { return __uint_as_float(x << 16); }
__device__ __forceinline__ float bf_hi(uint32_t x) { return __uint_as_float(x & 0xffff0000u); }

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
}

// 2^x by the SFU alone (MUFU.EX2, denormal results flushed to zero): fast_exp2() wraps the same
// instruction in a range check and two scalings for denormals, which a softmax weight never needs.
__device__ __forceinline__ float fast_exp2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Packed fp32 arithmetic of sm_100 (fma.rn.f32x2: two independent FMAs per instruction, operands in 64-bit registers).
__device__ __forceinline__ uint64_t f2pack(float lo, float hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void f2unpack(uint64_t v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ uint64_t ffma2(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
// the two bf16 of a 32-bit word as an fp32 pair (exact)
__device__ __forceinline__ uint64_t bf2_to_f2(uint32_t w) { return f2pack(bf_lo(w), bf_hi(w)); }

// erfc-based exact-GELU with ONE special-function instruction: Phi(-|x|) = 0.5 erfc(|x| / sqrt 2) = 2^P(|x|) with a
// degree-6 polynomial P fitted on [0, 10] (max |error| of the GELU 5e-8 in exact arithmetic, 5e-7 in fp32 --
// below the bf16 rounding of the result by four orders of magnitude); gelu(x) = max(x, 0) - |x| Phi(-|x|).
// P(a) = -0.9999930605 - 1.151201707 a - 0.4587709584 a^2 - 0.05341212449 a^3 + 8.080729771e-3 a^4
//        - 7.692237508e-4 a^5 + 3.309327859e-5 a^6, |x| clamped to 10 (beyond it Phi(-|x|) < 1e-23).
// Two of them at once on the packed fp32 pipe (fma.rn.f32x2: one instruction, two FMAs) -> one bf16x2 word.
__device__ __forceinline__ uint32_t gelu_erfc_x2(float x0, float x1) {
    const float a0 = fminf(fabsf(x0), 10.0f), a1 = fminf(fabsf(x1), 10.0f);
    const uint64_t ax = f2pack(a0, a1);
    uint64_t p = ffma2(f2pack(3.309327859e-05f, 3.309327859e-05f), ax, f2pack(-7.692237508e-04f, -7.692237508e-04f));
    p = ffma2(p, ax, f2pack(8.080729771e-03f, 8.080729771e-03f));
    p = ffma2(p, ax, f2pack(-5.341212449e-02f, -5.341212449e-02f));
    p = ffma2(p, ax, f2pack(-4.587709584e-01f, -4.587709584e-01f));
    p = ffma2(p, ax, f2pack(-1.151201707e+00f, -1.151201707e+00f));
    p = ffma2(p, ax, f2pack(-9.999930605e-01f, -9.999930605e-01f));
    float p0, p1, e0, e1;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(p0), "=f"(p1) : "l"(p));
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e0) : "f"(p0));
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e1) : "f"(p1));
    const uint64_t g = ffma2(f2pack(-a0, -a1), f2pack(e0, e1), f2pack(fmaxf(x0, 0.f), fmaxf(x1, 0.f)));
    float g0, g1;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(g0), "=f"(g1) : "l"(g));
    return pack_bf16(g0, g1);
}

// exact GELU, 0.5 x (1 + erf(x / sqrt 2))  (reading A5)
__device__ __forceinline__ float gelu_erf(float x) { return 0.5f * x * (1.0f + erff(x * 0.70710678118654752f)); }

// Shared-memory geometry (strides chosen so mma fragment accesses are bank-conflict free).
template <int D, int NT>
struct Geo {
    static constexpr int R = 8 * NT;          // rows per tile
    static constexpr int HS = D + 4;          // fp32 residual stream stride (words)
    static constexpr int AS = D + 8;          // bf16 activation stride (elements)
    static constexpr int QS = 3 * D + 4;      // fp32 q|k|v stride (words)
    static constexpr int FS = 4 * D + 8;      // bf16 FFN hidden stride (elements)
    static constexpr int KS2 = 2;             // K-splits of the W2 GEMM (= ring chunks per m-tile, fv_decode.cu)
    static constexpr size_t h_bytes = (size_t)R * HS * 4;
    static constexpr size_t a_bytes = (size_t)R * AS * 2;
    static constexpr size_t qkv_bytes = (size_t)R * QS * 4;
    static constexpr size_t hid_bytes = (size_t)R * FS * 2;
    static constexpr size_t part_bytes = (size_t)KS2 * R * HS * 4;
    static constexpr size_t big_bytes = (qkv_bytes > hid_bytes + part_bytes) ? qkv_bytes : hid_bytes + part_bytes;
    static constexpr size_t split_bytes = (size_t)16 * (D + 2 * (D / 8)) * 4;   // attention split partials
    static constexpr size_t misc_bytes = (size_t)R * (8 + 4 * 5);            // logq f64, logp, u, tok, b, t
    static constexpr size_t total = h_bytes + a_bytes + big_bytes + split_bytes + misc_bytes + 64;
};

// out[row][feat] = sum_k W[feat][k] * act[row][k] for one tile of 8*NT rows.
// W is pre-packed (fragment order), act is bf16 in shared memory with row stride `as`.
// Tasks (mt, ks) = (16 output features, one K-split) are dealt round-robin to the warps;
// epi(mt, ks, acc) receives acc[nt][4]: {(f, r), (f, r+1), (f+8, r), (f+8, r+1)} with
// f = 16 mt + lane/4 and r = 8 nt + 2 (lane%4).
// The weight stream comes from L2 (latency ~1 us under load) and nothing is reused, so the
// loads of up to TPB tasks (MAXL x 128-bit per lane) are issued before the first MMA: one L2
// round trip per GEMM phase instead of one per task.
template <int KT_TOTAL, int KSPLIT, int NT, int NW, int MAXL = 16, class Epi>
__device__ __forceinline__ void gemm_rows(const uint4* __restrict__ wp, int MT, const __nv_bfloat16* act, int as,
                                          int warp, int lane, Epi epi) {
    constexpr int KT = KT_TOTAL / KSPLIT;
    constexpr int KU = KT < MAXL ? KT : MAXL;
    constexpr int TPB = (MAXL / KU) < 4 ? (MAXL / KU) : 4;
    const int g = lane >> 2, c = lane & 3;
    const int total = MT * KSPLIT;
    for (int task0 = warp; task0 < total; task0 += NW * TPB) {
        uint4 a[TPB][KU];
#pragma unroll
        for (int tb = 0; tb < TPB; ++tb) {
            const int task = task0 + tb * NW;
            if (task < total) {
                const int mt = task / KSPLIT, ks = task - mt * KSPLIT;
                const uint4* w = wp + ((size_t)mt * KT_TOTAL + ks * KT) * 32 + lane;
#pragma unroll
                for (int u = 0; u < KU; ++u) a[tb][u] = ldg_w(w + u * 32);
            }
        }
#pragma unroll
        for (int tb = 0; tb < TPB; ++tb) {
            const int task = task0 + tb * NW;
            if (task < total) {
                const int mt = task / KSPLIT, ks = task - mt * KSPLIT;
                float acc[NT][4];
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) acc[nt][0] = acc[nt][1] = acc[nt][2] = acc[nt][3] = 0.f;
                const uint4* w = wp + ((size_t)mt * KT_TOTAL + ks * KT) * 32 + lane;
                const __nv_bfloat16* ab = act + g * as + ks * KT * 16 + 2 * c;
#pragma unroll 1
                for (int k0 = 0; k0 < KT; k0 += KU) {
                    if (k0 > 0) {
#pragma unroll
                        for (int u = 0; u < KU; ++u) a[tb][u] = ldg_w(w + (k0 + u) * 32);
                    }
#pragma unroll
                    for (int u = 0; u < KU; ++u) {
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) {
                            const __nv_bfloat16* p = ab + nt * 8 * as + (k0 + u) * 16;
                            mma_bf16(acc[nt], a[tb][u], lds32(p), lds32(p + 8));
                        }
                    }
                }
                epi(mt, ks, acc);
            }
        }
    }
}

// LayerNorm of one row held in shared memory (fp32), one warp per row: mean, biased variance,
// eps inside the sqrt, affine (reading A6).  Writes bf16 to `out`; if `replace` the fp32 row is
// overwritten with the normalised value (ln2_style 1, Alg. 1 l.5).
// SM: gam / bet point to shared memory (plain loads) instead of global memory (read-only path).
template <int D, bool SM = false>
__device__ __forceinline__ void ln_row(float* hrow, const float* __restrict__ gam, const float* __restrict__ bet,
                                       float eps, bool replace, __nv_bfloat16* out, int lane) {
    constexpr int E = D / 32;
    float x[E];
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < E; ++j) { x[j] = hrow[lane * E + j]; s += x[j]; }
    const float mean = warp_sum(s) * (1.0f / D);
    float v = 0.f;
#pragma unroll
    for (int j = 0; j < E; ++j) { const float dlt = x[j] - mean; v += dlt * dlt; }
    const float rstd = rsqrtf(warp_sum(v) * (1.0f / D) + eps);
#pragma unroll
    for (int j = 0; j < E; ++j) {
        const int i = lane * E + j;
        const float y = SM ? (x[j] - mean) * rstd * gam[i] + bet[i] : (x[j] - mean) * rstd * __ldg(gam + i) + __ldg(bet + i);
        out[i] = __float2bfloat16_rn(y);
        if (replace) hrow[i] = y;
    }
}

// Masked gather attention for ONE query row against entries [e_begin, e_end) of its CSR mask
// row (Eq. 3; mask Eq. S1 l.555 generalised to an index list).
// Lane layout: a KV row is 2D bf16 = K[D] | V[D]; LPR = D/8 lanes cover K (16 B each) and the
// same lanes fetch the matching 16 B of V, so a warp handles RPI = 32/LPR rows per iteration.
// A head spans LPH = DH/8 adjacent lanes; its score is completed by shfl.xor over them.
// Online softmax in base 2 (q is pre-scaled by log2(e)/sqrt(d_h)); state (m, l, acc[8]) is per
// lane and merged across the RPI row groups at the end, so every lane returns the result.
template <int D, int DH>
__device__ __forceinline__ void attend_range(const float* qrow, const __nv_bfloat16* kv_sl, const int32_t* __restrict__ cols,
                                             int e_begin, int e_end, int lane, float& m_out, float& l_out,
                                             float (&acc)[8]) {
    constexpr int LPR = D / 8, RPI = 32 / LPR, LPH = DH / 8, U = 4;
    const int rg = lane / LPR, sub = lane % LPR;
    const float qs = kLog2e * rsqrtf((float)DH);
    float q[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) q[j] = qrow[sub * 8 + j] * qs;
    float m = -1e30f, l = 0.f;
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[j] = 0.f;
    const char* base = reinterpret_cast<const char*>(kv_sl) + sub * 16;
    for (int e0 = e_begin; e0 < e_end; e0 += RPI * U) {
        uint4 kk[U], vv[U];
        bool ok[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int e = e0 + u * RPI + rg;
            ok[u] = e < e_end;
            const int pos = __ldg(cols + (ok[u] ? e : e_begin));
            const char* p = base + (size_t)pos * (4 * D);
            kk[u] = ld_kv(p);
            vv[u] = ld_kv(p + 2 * D);
        }
        float s[U];
        float mx = m;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            float d = q[0] * bf_lo(kk[u].x) + q[1] * bf_hi(kk[u].x);
            d += q[2] * bf_lo(kk[u].y) + q[3] * bf_hi(kk[u].y);
            d += q[4] * bf_lo(kk[u].z) + q[5] * bf_hi(kk[u].z);
            d += q[6] * bf_lo(kk[u].w) + q[7] * bf_hi(kk[u].w);
#pragma unroll
            for (int o = 1; o < LPH; o <<= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
            s[u] = ok[u] ? d : -INFINITY;
            mx = fmaxf(mx, s[u]);
        }
        const float corr = fast_exp2(m - mx);
        m = mx;
        l *= corr;
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[j] *= corr;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const float p = fast_exp2(s[u] - mx);
            l += p;
            acc[0] += p * bf_lo(vv[u].x); acc[1] += p * bf_hi(vv[u].x);
            acc[2] += p * bf_lo(vv[u].y); acc[3] += p * bf_hi(vv[u].y);
            acc[4] += p * bf_lo(vv[u].z); acc[5] += p * bf_hi(vv[u].z);
            acc[6] += p * bf_lo(vv[u].w); acc[7] += p * bf_hi(vv[u].w);
        }
    }
#pragma unroll
    for (int o = LPR; o < 32; o <<= 1) {       // merge the RPI row groups
        const float m2 = __shfl_xor_sync(0xffffffffu, m, o);
        const float l2 = __shfl_xor_sync(0xffffffffu, l, o);
        const float mx = fmaxf(m, m2);
        const float c1 = fast_exp2(m - mx), c2 = fast_exp2(m2 - mx);
        l = l * c1 + l2 * c2;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const float a2 = __shfl_xor_sync(0xffffffffu, acc[j], o);
            acc[j] = acc[j] * c1 + a2 * c2;
        }
        m = mx;
    }
    m_out = m;
    l_out = l;
}


}  // namespace fvdev
