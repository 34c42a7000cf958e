// fv_ring.cuh -- pieces shared by the two samplers of fv_sample (fv_decode.cu: one CTA owns its samples for
// all layers, weights streamed; fv_chain.cu: a cluster of n_layers CTAs, one layer's weights resident per CTA):
// mbarrier / TMA bulk-copy / cluster (distributed shared memory) wrappers, the shared-memory KV ring protocol
// (producer arms chunks in order, one consumer warp per chunk) and the online-softmax update of one query row
// with the rows of one ring chunk (Eq. 3).
#pragma once
#include "fv_device.cuh"
#include "fv_umma.cuh"

namespace fvring {
using namespace fvdev;

constexpr int NWC = 16;                       // compute warps of both sampler kernels
constexpr size_t SMEM_MAX = 232448;           // 227 KB per CTA on sm_100

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_n(uint64_t* bar, uint32_t n) {       // n arrivals at once
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(n) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    const uint32_t addr = smem_u32(bar);
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}\n"
            : "=r"(done) : "r"(addr), "r"(parity) : "memory");
    } while (!done);
}
// One bounded probe of a phase (the hardware suspends the thread for a short, implementation-defined time).
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}\n"
        : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return done != 0;
}
// Non-blocking probe (mbarrier.test_wait never suspends the thread).
__device__ __forceinline__ bool mbar_test_nb(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}\n"
        : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return done != 0;
}
// TMA 1-D bulk copy global -> shared, completion counted in bytes on an mbarrier.
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// The same with an L2 eviction policy (createpolicy) attached to the read.
__device__ __forceinline__ void bulk_g2s_hint(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;\n"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
// ---- 2-CTA cluster plumbing (distributed shared memory) -------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;\n" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}
__device__ __forceinline__ uint32_t map_to_peer(uint32_t saddr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_peer128(uint32_t raddr, uint4 v) {
    asm volatile("st.shared::cluster.v4.b32 [%0], {%1,%2,%3,%4};\n" ::"r"(raddr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void mbar_arrive_peer(uint32_t raddr) {
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];\n" ::"r"(raddr) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint64_t* bar, uint32_t parity) {
    const uint32_t addr = smem_u32(bar);
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}\n"
            : "=r"(done) : "r"(addr), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void cbar() { asm volatile("bar.sync 1, %0;\n" ::"n"(NWC * 32) : "memory"); }
__device__ __forceinline__ int ld_acquire_s32(const int* p) {
    int v;
    asm volatile("ld.acquire.cta.shared.s32 %0, [%1];\n" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_s32(int* p, int v) {
    asm volatile("st.release.cta.shared.s32 [%0], %1;\n" ::"r"(smem_u32(p)), "r"(v) : "memory");
}

// Online-softmax update of one query row with the `rows` KV rows of one ring chunk (Eq. 3,
// PAPER.md:102).  Lane layout as attend_range (fv_device.cuh): LPR = D/8 lanes cover one K row
// with 128-bit shared loads and the matching 16 B of V; RPI = 32/LPR rows per iteration.
// The phase is issue-bound (about 25 instructions per row and warp before, two thirds of them the
// bf16 unpacking and the FMAs): scores and the P V update run on the packed fp32 pipe, even and odd
// features in the two halves of a register pair, which takes a third of the FMA instructions out.
// NS warps share a query row by HEADS (NS = 2: each warp takes D / 2 features, i.e. whole heads, of every row of the
// chunk -- nothing to merge between the warps afterwards); then LPR = D / 8 / NS lanes cover a warp's part of a row and
// `base` already points at that part.
template <int D, int DH, int UU, int NS>
__device__ __forceinline__ void attend_rows(const unsigned char* base, int i0, int rows, const uint64_t (&q2)[4], int rg,
                                            float& m, float& l, uint64_t (&a2)[4]) {
    constexpr int LPR = D / 8 / NS, RPI = 32 / LPR, LPH = DH / 8;
    static_assert(LPR >= LPH && LPR % LPH == 0, "a warp's part of a row holds whole heads");
    uint4 kk[UU], vv[UU];
    bool ok[UU];
#pragma unroll
    for (int u = 0; u < UU; ++u) {
        const int row = i0 + u * RPI + rg;
        ok[u] = row < rows;
        const unsigned char* p = base + (size_t)(ok[u] ? row : 0) * (4 * D);
        kk[u] = *reinterpret_cast<const uint4*>(p);
        vv[u] = *reinterpret_cast<const uint4*>(p + 2 * D);
    }
    float s[UU];
    float mx = m;
#pragma unroll
    for (int u = 0; u < UU; ++u) {
        uint64_t d2 = ffma2(q2[0], bf2_to_f2(kk[u].x), 0ull);
        d2 = ffma2(q2[1], bf2_to_f2(kk[u].y), d2);
        d2 = ffma2(q2[2], bf2_to_f2(kk[u].z), d2);
        d2 = ffma2(q2[3], bf2_to_f2(kk[u].w), d2);
        float de, dodd;
        f2unpack(d2, de, dodd);
        float d = de + dodd;
#pragma unroll
        for (int o = 1; o < LPH; o <<= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
        s[u] = ok[u] ? d : -INFINITY;
        mx = fmaxf(mx, s[u]);
    }
    const float corr = fast_exp2(m - mx);
    m = mx;
    l *= corr;
    const uint64_t c2 = f2pack(corr, corr);
#pragma unroll
    for (int j = 0; j < 4; ++j) a2[j] = ffma2(a2[j], c2, 0ull);
#pragma unroll
    for (int u = 0; u < UU; ++u) {
        const float p = fast_exp2(s[u] - mx);
        l += p;
        const uint64_t p2 = f2pack(p, p);
        a2[0] = ffma2(p2, bf2_to_f2(vv[u].x), a2[0]);
        a2[1] = ffma2(p2, bf2_to_f2(vv[u].y), a2[1]);
        a2[2] = ffma2(p2, bf2_to_f2(vv[u].z), a2[2]);
        a2[3] = ffma2(p2, bf2_to_f2(vv[u].w), a2[3]);
    }
}

// The same update with ONE row per row group whose K / V words the lane already holds in registers (rows fv_decode.cu
// loads straight from the pool; `ok` false = this row group has none).
template <int DH>
__device__ __forceinline__ void attend_direct(const uint4& kk, const uint4& vv, bool ok, const float (&q)[8],
                                              float& m, float& l, float (&acc)[8]) {
    constexpr int LPH = DH / 8;
    uint64_t d2 = ffma2(f2pack(q[0], q[1]), bf2_to_f2(kk.x), 0ull);
    d2 = ffma2(f2pack(q[2], q[3]), bf2_to_f2(kk.y), d2);
    d2 = ffma2(f2pack(q[4], q[5]), bf2_to_f2(kk.z), d2);
    d2 = ffma2(f2pack(q[6], q[7]), bf2_to_f2(kk.w), d2);
    float de, dodd;
    f2unpack(d2, de, dodd);
    float d = de + dodd;
#pragma unroll
    for (int o = 1; o < LPH; o <<= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
    const float s = ok ? d : -INFINITY;
    const float mx = fmaxf(m, s);
    const float corr = fast_exp2(m - mx), p = fast_exp2(s - mx);
    m = mx;
    l = l * corr + p;
    const uint32_t w[4] = {vv.x, vv.y, vv.z, vv.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        acc[2 * j] = acc[2 * j] * corr + p * bf_lo(w[j]);
        acc[2 * j + 1] = acc[2 * j + 1] * corr + p * bf_hi(w[j]);
    }
}

// Full groups of U row sets, then the remaining rows one set (RPI rows) at a time: a ragged tail chunk of two rows
// costs a quarter of a group instead of a whole one (cfg5: the fifth chunk of every sample holds 2 of 16 rows).
template <int D, int DH, int CH, int NS = 1>
__device__ __forceinline__ void attend_chunk(const unsigned char* chunk, int rows, const float (&q)[8], int rg, int sub,
                                             float& m, float& l, float (&acc)[8]) {
    constexpr int LPR = D / 8 / NS, RPI = 32 / LPR;
    constexpr int ITER = (CH + RPI - 1) / RPI, U = ITER < 4 ? ITER : 4;
    const unsigned char* base = chunk + sub * 16;
    const uint64_t q2[4] = {f2pack(q[0], q[1]), f2pack(q[2], q[3]), f2pack(q[4], q[5]), f2pack(q[6], q[7])};
    uint64_t a2[4] = {f2pack(acc[0], acc[1]), f2pack(acc[2], acc[3]), f2pack(acc[4], acc[5]), f2pack(acc[6], acc[7])};
    int i0 = 0;
    for (; i0 + RPI * U <= rows; i0 += RPI * U) attend_rows<D, DH, U, NS>(base, i0, rows, q2, rg, m, l, a2);
    for (; i0 < rows; i0 += RPI) attend_rows<D, DH, 1, NS>(base, i0, rows, q2, rg, m, l, a2);
#pragma unroll
    for (int j = 0; j < 4; ++j) f2unpack(a2[j], acc[2 * j], acc[2 * j + 1]);
}

// LayerNorm of one fp32 row of 128 features in shared memory (reading A6), one warp per row, written as row r of
// the [NB x 128] K-major SWIZZLE_128B B tile of a swap-AB tcgen05 GEMM (two K-blocks of NB rows x 128 B).
template <int NB>
__device__ __forceinline__ void ln_row_btile(float* hrow, const float* __restrict__ gam, const float* __restrict__ bet,
                                             float eps, bool replace, unsigned char* btile, int r, int lane) {
    constexpr int DD = 128;
    const float4 x = *reinterpret_cast<const float4*>(hrow + lane * 4);
    const float mean = warp_sum(x.x + x.y + x.z + x.w) * (1.0f / DD);
    const float d0 = x.x - mean, d1 = x.y - mean, d2 = x.z - mean, d3 = x.w - mean;
    const float rstd = rsqrtf(warp_sum(d0 * d0 + d1 * d1 + d2 * d2 + d3 * d3) * (1.0f / DD) + eps);
    const float4 g = __ldg(reinterpret_cast<const float4*>(gam) + lane), b = __ldg(reinterpret_cast<const float4*>(bet) + lane);
    const float y0 = d0 * rstd * g.x + b.x, y1 = d1 * rstd * g.y + b.y, y2 = d2 * rstd * g.z + b.z, y3 = d3 * rstd * g.w + b.w;
    const int i0 = lane * 4, kb = i0 >> 6, c = (i0 & 63) >> 3;
    uint2 pk;
    pk.x = pack_bf16(y0, y1);
    pk.y = pack_bf16(y2, y3);
    *reinterpret_cast<uint2*>(btile + kb * (NB * 128) + umma::sw128_chunk(r, c) + (i0 & 7) * 2) = pk;
    if (replace) *reinterpret_cast<float4*>(hrow + lane * 4) = make_float4(y0, y1, y2, y3);
}

// Consumer side of a ring chunk: wait until the producer has armed this round of the slot (a
// parity wait can only tell a phase from its predecessor, and another warp may still own the
// slot's previous round), then wait for the bytes.
struct RingCtx {
    unsigned char* ring;
    uint64_t* bar_full;
    uint64_t* bar_empty;
    int* issued;
};
template <int NSLOT, int CHUNK_BYTES>
__device__ __forceinline__ unsigned char* ring_acquire(const RingCtx& rc, uint32_t sq, uint32_t& slot) {
    slot = sq % NSLOT;
    const uint32_t par = (sq / NSLOT) & 1u;
    while ((int)((uint32_t)ld_acquire_s32(rc.issued) - sq) <= 0) __nanosleep(20);
    mbar_wait(rc.bar_full + slot, par);
    return rc.ring + (size_t)slot * CHUNK_BYTES;
}
__device__ __forceinline__ void ring_release(const RingCtx& rc, uint32_t slot, int lane, uint32_t arrivals = 1) {
    // The slot is refilled by cp.async.bulk (async proxy): order this warp's generic-proxy reads of
    // it before that write.  Without the fence a refill could overtake the reads (seen as run-to-run
    // differences of ~1e-4 in both samples of a CTA at one step, 15 of 16 fresh-model runs).
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    __syncwarp();
    if (lane == 0) mbar_arrive_n(rc.bar_empty + slot, arrivals);
}

// The same release without the proxy fence, for a warp whose reads of the slot have all been CONSUMED: `h` must be computed
// (in every lane) from results of arithmetic that used every value the lane loaded from the slot.  The hazard the fence
// guards against is the arrive (issued to the barrier unit, SYNCS) overtaking shared-memory loads still in flight, so that
// the refill lands before they are performed; a load whose value has been used is performed.  The vote cannot issue before
// h is ready in all lanes and the arrive takes its count from the vote's result, so the arrive issues after every such
// load has returned -- in SASS, not only in program order (the compare is never true in practice and both counts are equal).
__device__ __forceinline__ void ring_release_dep(const RingCtx& rc, uint32_t slot, int lane, uint32_t arrivals, uint32_t h) {
    uint32_t same;
    asm volatile("mov.u32 %0, %1;" : "=r"(same) : "r"(arrivals));
    const bool never = __any_sync(0xffffffffu, h == 0x9E3779B9u);
    if (lane == 0) mbar_arrive_n(rc.bar_empty + slot, never ? arrivals : same);
}

}  // namespace fvring
