// fv_decode.cu -- the persistent KV-cached sampler of fv_sample (Alg. 2) for sm_100a.
//
// A CTA owns a group of S <= 8*NT samples for all N steps (samples are independent, l.125, so
// CTAs never communicate).  Per step t and layer: LN1 -> QKV -> KV append -> masked attention
// over the rows A(t) of the CSR mask -> (W_O) -> LN2 -> FFN -> residual; then the sigmoid head,
// the Bernoulli draw from the caller's uniform and the log q update.
//
// The streams are decoupled from the compute warps.  The mask is static, so every KV row a step will
// need -- except the row the step itself appends -- is known long before; one PRODUCER warp walks
// (t, layer) in the consumers' order and streams ONE ordered sequence of 8 KB chunks into a shared
// memory ring with cp.async.bulk (TMA 1-D bulk copies) completing on mbarriers: the layer's W_qkv,
// the KV rows the mask names for every sample (runs of consecutive positions merged into one copy by
// the host plan), W_o, W_1, W_2.  The 16 COMPUTE warps read K/V and the mma.sync A fragments from
// shared memory.  Row t itself is attended from the shared memory of the step that produced it
// (rounded to bf16 exactly as the pool stores it).
// What paces the kernel is the latency chain "consumer frees slots -> producer round -> copies land" (DESIGN.md 6.1,
// profiles/r03_fv_sample.md), so: weight chunks travel two per bulk copy; isolated key rows (runs of one row) bypass the ring
// and are loaded by the attention warps (plan d_* of fv_internal.h); the producer maps chunk -> (sample, chunk) without
// integer divisions; slots are released through a data dependency instead of a proxy fence (ring_release_dep); the two
// warps of a sample split its query row by heads (no partial results, no combine phase); a layer's small parameters are
// staged in shared memory by warps that would otherwise wait.
// Optional (FLASHVAN_DECODE=cluster): 2-CTA clusters in which each CTA streams only its half of
// W_1/W_2 and applies it to the rows of both CTAs, exchanging LN2 rows and partial sums through
// distributed shared memory (correct, measured slower: DESIGN.md 6.1).
#include "fv_ring.cuh"

namespace {
using namespace fvring;

constexpr int NTHREADS = NWC * 32 + 32;       // compute warps + the producer warp
#ifndef FV_DEC_WG
#define FV_DEC_WG 2
#endif
constexpr int GEMM_MAXL = 8;                  // 128-bit weight loads in flight per lane when the weights come by LDG (d = 256)

// CL = the CTA is one half of a 2-CTA cluster that splits the FFN (see the kernel header).
template <int D, int NT, bool CL = false>
struct DecGeo {
    using G = Geo<D, NT>;
    // cluster mode: FFN over the 2R rows of both CTAs, hidden half (2D columns) per CTA
    static constexpr int R2 = 2 * G::R, FS2 = 2 * D + 8;
    // q stays fp32; k|v of the step are kept as the bf16 the pool stores (append = plain copy)
    static constexpr int QS2 = D + 4, KVS = 2 * D + 8;
    static constexpr size_t q_bytes = (size_t)G::R * QS2 * 4;
    static constexpr size_t qkv_bytes = q_bytes + (size_t)G::R * KVS * 2;
    static constexpr size_t hid2_bytes = (size_t)R2 * FS2 * 2;
    static constexpr size_t part2_bytes = (size_t)R2 * G::HS * 4;
    // the FFN2 partial sums reuse the attention-split buffer when they fit (both are dead by then)
    // attention-split partials exist only when several warps share a query row (R <= 8)
    static constexpr size_t split_bytes = (NWC / G::R > 1) ? G::split_bytes : 0;
    // W2 partial sums: with >= 16 rows per CTA a warp takes whole m-tiles and accumulates straight into
    // the residual stream (gemm_ring_kparts: no buffer, 33 KB more ring at 32 rows); with 8 rows the two
    // K-halves go to two warps (measured faster there) and their partial sums reuse the attention-split
    // buffer, which is dead by then
    static constexpr bool NO_PART = !CL && D <= 128 && NT >= 2;
    static constexpr bool PART_IN_SPLIT = !CL && !NO_PART && G::part_bytes <= split_bytes;
    static constexpr size_t big_bytes = CL ? (qkv_bytes > hid2_bytes + part2_bytes ? qkv_bytes : hid2_bytes + part2_bytes)
                                      : (!(NO_PART || PART_IN_SPLIT)
                                             ? (qkv_bytes > G::hid_bytes + G::part_bytes ? qkv_bytes : G::hid_bytes + G::part_bytes)
                                             : (qkv_bytes > G::hid_bytes ? qkv_bytes : G::hid_bytes));
    static constexpr size_t xa_bytes = CL ? (size_t)R2 * G::AS * 2 : 0;     // LN2 activations of both CTAs (peer-written)
    static constexpr size_t xp_bytes = CL ? (size_t)G::R * G::HS * 4 : 0;   // peer's FFN2 partial sums for my rows
    // the current layer's LayerNorm gains / biases and GEMM biases (FvLayerDev::par), staged by warps that would otherwise
    // wait: as __ldg operands they cost an L2 round trip in every phase (L1 is ~28 KB next to this carve-out)
    static constexpr int PAR_E = 5 * D, PAR_L = 8 * D;     // floats used up to the QKV epilogue / after it
    static constexpr size_t par_bytes = (size_t)(PAR_E + PAR_L) * 4;
    static constexpr size_t geo_total = G::total - G::big_bytes - G::split_bytes + big_bytes + split_bytes + par_bytes + xa_bytes + xp_bytes;
    static constexpr int CH = fv_ring_ch(D);              // KV rows per ring chunk (host plan agrees)
    static constexpr int ROW_BYTES = 4 * D;               // K[D] | V[D] in bf16
    static constexpr int CHUNK_BYTES = CH * ROW_BYTES;
    static constexpr size_t fixed = (geo_total + 127) / 128 * 128;
    static constexpr int TAB_C = 48, TAB_R = 48;          // per-step copy plan staged in smem (x2: t, t+1)
    static constexpr size_t bar_bytes = 1024 + 2 * (TAB_C * 4 + TAB_R * 8);   // mbarriers (2 x 60 + 2), counters, plans
    static constexpr int NSLOT_RAW = (int)((SMEM_MAX - fixed - bar_bytes) / CHUNK_BYTES);
    static constexpr int NSLOT_CAP = 60;
    // Weight chunks travel in groups of WG consecutive chunks = ONE bulk copy of WG * CHUNK_BYTES into WG adjacent slots
    // (the TMA unit costs ~30 ns per copy + 4.4 ns per KB: 8 KB copies feed an SM with 124 GB/s, 16 KB with 163 GB/s, and
    // the stream is what the compute warps wait for).  Groups never wrap: NSLOT is a multiple of WG and every section of
    // the chunk sequence (a weight matrix, the KV chunks of a layer-step padded with empty chunks) is one too.
    static constexpr int WG = (!CL && D == 128) ? FV_DEC_WG : 1;
    static constexpr int NSLOT = (NSLOT_RAW > NSLOT_CAP ? NSLOT_CAP : NSLOT_RAW) / WG * WG;
    static constexpr size_t total = fixed + bar_bytes + (size_t)NSLOT * CHUNK_BYTES;
    // GEMM weights stream through the same ring (D <= 128): a chunk is CHUNK_BYTES of the packed
    // image = TPCH 16x16 tiles = whole m-tiles (K = D) or one K-part of an m-tile (K = 4D).
    static constexpr bool WRING = D <= 128;
    static constexpr int TPCH = CHUNK_BYTES / 512;
    static constexpr int NQ = (3 * D / 16) * (D / 16) / TPCH;     // W_qkv chunks
    static constexpr int NO = (D / 16) * (D / 16) / TPCH;         // W_o
    static constexpr int N1 = (4 * D / 16) * (D / 16) / TPCH;     // W_1
    static constexpr int N2 = (D / 16) * (4 * D / 16) / TPCH;     // W_2
    static_assert(NSLOT >= 2, "KV ring needs at least two chunks");
};


// Weight chunk sq of a group of WG chunks that arrived with one bulk copy: the bytes complete on the full barrier of
// the group's FIRST slot (sections start at multiples of WG, so sq % WG is the chunk's place in its group).
template <int NSLOT, int CHUNK_BYTES, int WG>
__device__ __forceinline__ unsigned char* ring_acquire_w(const RingCtx& rc, uint32_t sq, uint32_t& slot) {
    if constexpr (WG == 1) return ring_acquire<NSLOT, CHUNK_BYTES>(rc, sq, slot);
    slot = sq % NSLOT;
    const uint32_t s0 = sq - sq % WG;
    while ((int)((uint32_t)ld_acquire_s32(rc.issued) - sq) <= 0) __nanosleep(20);
    mbar_wait(rc.bar_full + s0 % NSLOT, (s0 / NSLOT) & 1u);
    return rc.ring + (size_t)slot * CHUNK_BYTES;
}

// GEMM over one tile of 8*NT rows with the weights taken from ring chunks (same contract as
// gemm_rows).  Chunk j of a matrix holds TPCH consecutive 16x16 tiles of its packed image:
// MPC whole m-tiles when K fits a chunk, else K-part (j % KSP) of m-tile j / KSP.  Warp w
// consumes chunks w, w + NWC, ... (ring order), A fragments by conflict-free 128-bit LDS.
template <int KT_TOTAL, int NT, int TPCH, int NSLOT, int CHUNK_BYTES, int WG, int EC, class Epi>
__device__ __forceinline__ void gemm_ring(const RingCtx& rc, int nchunks, uint32_t seq0, const __nv_bfloat16* act,
                                          int as, int warp, int lane, Epi epi) {
    constexpr bool SPLITK = KT_TOTAL > TPCH;
    constexpr int KSP = SPLITK ? KT_TOTAL / TPCH : 1;
    constexpr int MPC = SPLITK ? 1 : TPCH / KT_TOTAL;
    constexpr int KT = SPLITK ? TPCH : KT_TOTAL;
    const int g = lane >> 2, c = lane & 3;
    for (int j = warp; j < nchunks; j += NWC) {
        uint32_t slot;
        const uint4* wsm = reinterpret_cast<const uint4*>(ring_acquire_w<NSLOT, CHUNK_BYTES, WG>(rc, seq0 + (uint32_t)j, slot)) + lane;
        const int ks = SPLITK ? j - (j / KSP) * KSP : 0;
        const __nv_bfloat16* ab = act + g * as + ks * KT * 16 + 2 * c;
        // k outer, m-tiles inner: the activation fragments of a k-step are read once and feed MPC (K = D)
        // or two (K-part of W2: even / odd k-steps) independent accumulator chains
        constexpr int NCH = SPLITK ? 2 : MPC;
        float acc[NCH][NT][4];
#pragma unroll
        for (int q = 0; q < NCH; ++q)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) acc[q][nt][0] = acc[q][nt][1] = acc[q][nt][2] = acc[q][nt][3] = 0.f;
#pragma unroll
        for (int kt = 0; kt < KT; ++kt) {
            uint32_t b0[NT], b1[NT];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
                const __nv_bfloat16* p = ab + nt * 8 * as + kt * 16;
                b0[nt] = lds32(p); b1[nt] = lds32(p + 8);
            }
            if constexpr (SPLITK) {
                const uint4 aw = wsm[kt * 32];
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) mma_bf16(acc[kt & 1][nt], aw, b0[nt], b1[nt]);
            } else {
#pragma unroll
                for (int mi = 0; mi < MPC; ++mi) {
                    const uint4 aw = wsm[(mi * KT + kt) * 32];
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) mma_bf16(acc[mi][nt], aw, b0[nt], b1[nt]);
                }
            }
        }
        {   // every A fragment read from the slot has fed an MMA of one of these accumulators
            uint32_t h = 0;
#pragma unroll
            for (int q = 0; q < NCH; ++q)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) h ^= __float_as_uint(acc[q][nt][0]);
            ring_release_dep(rc, slot, lane, EC, h);
        }
        if constexpr (SPLITK) {
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int e = 0; e < 4; ++e) acc[0][nt][e] += acc[1][nt][e];
            epi(j / KSP, ks, acc[0]);
        } else {
#pragma unroll
            for (int mi = 0; mi < MPC; ++mi) epi(j * MPC + mi, 0, acc[mi]);
        }
    }
}

// W2 GEMM (K = 4D > one chunk) with all KSP K-parts of an m-tile consumed by the SAME warp, one after the
// other (ring order), into one accumulator: no partial-sum buffer and no separate reduction phase --
// epi(mt, acc) applies bias and residual directly.
template <int KT_TOTAL, int NT, int TPCH, int NSLOT, int CHUNK_BYTES, int WG, int EC, class Epi>
__device__ __forceinline__ void gemm_ring_kparts(const RingCtx& rc, int n_mtiles, uint32_t seq0, const __nv_bfloat16* act,
                                                 int as, int warp, int lane, Epi epi) {
    static_assert(KT_TOTAL % TPCH == 0 && KT_TOTAL > TPCH, "K must span several chunks");
    constexpr int KSP = KT_TOTAL / TPCH, KT = TPCH;
    const int g = lane >> 2, c = lane & 3;
    for (int mt = warp; mt < n_mtiles; mt += NWC) {
        float acc[2][NT][4];                         // even / odd k-steps: two independent MMA chains
#pragma unroll
        for (int q = 0; q < 2; ++q)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) acc[q][nt][0] = acc[q][nt][1] = acc[q][nt][2] = acc[q][nt][3] = 0.f;
#pragma unroll 1
        for (int ks = 0; ks < KSP; ++ks) {
            uint32_t slot;
            const uint4* wsm = reinterpret_cast<const uint4*>(
                ring_acquire_w<NSLOT, CHUNK_BYTES, WG>(rc, seq0 + (uint32_t)(mt * KSP + ks), slot)) + lane;
            const __nv_bfloat16* ab = act + g * as + ks * KT * 16 + 2 * c;
#pragma unroll
            for (int kt = 0; kt < KT; ++kt) {
                const uint4 aw = wsm[kt * 32];
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    const __nv_bfloat16* p = ab + nt * 8 * as + kt * 16;
                    mma_bf16(acc[kt & 1][nt], aw, lds32(p), lds32(p + 8));
                }
            }
            {
                uint32_t h = 0;
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) h ^= __float_as_uint(acc[0][nt][0]) ^ __float_as_uint(acc[1][nt][0]);
                ring_release_dep(rc, slot, lane, EC, h);
            }
        }
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int e = 0; e < 4; ++e) acc[0][nt][e] += acc[1][nt][e];
        epi(mt, acc[0]);
    }
}

template <int D, int DH, int NT, bool CL>
__global__ void __launch_bounds__(NTHREADS, 1)
fv_decode_kernel(const __grid_constant__ FvModelDev m, const __grid_constant__ FvForwardArgs a) {
    using G = Geo<D, NT>;
    using DG = DecGeo<D, NT, CL>;
    [[maybe_unused]] constexpr int R2 = DG::R2, FS2 = DG::FS2, NT2 = 2 * NT;
    constexpr int R = G::R, HS = G::HS, AS = G::AS, FS = G::FS, KS2 = G::KS2;
    constexpr int NSPLIT = (NWC / R) > 1 ? (NWC / R) : 1;    // warps cooperating on one query row
    constexpr int LPR = D / 8, LPH = DH / 8;
    constexpr int SPS = D + 2 * LPR;                          // floats per split-partial slot
    constexpr int GR = NWC / NSPLIT;                          // samples attended at the same time
    constexpr int CH = DG::CH, NSLOT = DG::NSLOT, NSLOT_MAX = DG::NSLOT;
    static_assert(R * NSPLIT <= 16 || NSPLIT == 1, "split slots");

    extern __shared__ __align__(128) unsigned char smem[];
    float* sh_h = reinterpret_cast<float*>(smem);
    __nv_bfloat16* sh_a = reinterpret_cast<__nv_bfloat16*>(smem + G::h_bytes);
    unsigned char* big = smem + G::h_bytes + G::a_bytes;
    float* sh_q = reinterpret_cast<float*>(big);
    __nv_bfloat16* sh_kv = reinterpret_cast<__nv_bfloat16*>(big + DG::q_bytes);
    constexpr int QS2 = DG::QS2, KVS = DG::KVS;
    __nv_bfloat16* sh_hid = reinterpret_cast<__nv_bfloat16*>(big);
    float* sh_split = reinterpret_cast<float*>(big + DG::big_bytes);
    [[maybe_unused]] float* sh_part = DG::PART_IN_SPLIT ? sh_split     // (unused if NO_PART)
                                                        : reinterpret_cast<float*>(big + (CL ? DG::hid2_bytes : G::hid_bytes));
    double* sh_logq = reinterpret_cast<double*>(big + DG::big_bytes + DG::split_bytes);
    float* sh_logp = reinterpret_cast<float*>(sh_logq + R);
    float* sh_u = sh_logp + R;
    int* sh_tok = reinterpret_cast<int*>(sh_u + R);
    // cluster exchange buffers sit at the end of the fixed region (the peer CTA writes them)
    __nv_bfloat16* sh_a2 = reinterpret_cast<__nv_bfloat16*>(smem + DG::fixed - DG::xa_bytes - DG::xp_bytes);
    float* sh_xp = reinterpret_cast<float*>(smem + DG::fixed - DG::xp_bytes);
    float* sh_par = reinterpret_cast<float*>(smem + DG::fixed - DG::xa_bytes - DG::xp_bytes - DG::par_bytes);
    uint64_t* bar_full = reinterpret_cast<uint64_t*>(smem + DG::fixed);
    uint64_t* bar_empty = bar_full + NSLOT_MAX;
    int* sh_app = reinterpret_cast<int*>(bar_empty + NSLOT_MAX);   // KV appends published so far
    int* sh_issued = sh_app + 1;                                   // ring chunks armed so far
    uint64_t* bar_x = reinterpret_cast<uint64_t*>(sh_app + 2);     // [2] cluster exchange barriers (LN2 rows, partials)
    int32_t* tab_c = reinterpret_cast<int32_t*>(smem + DG::fixed + 1024);
    int2* tab_r = reinterpret_cast<int2*>(tab_c + 2 * DG::TAB_C);
    unsigned char* ring = smem + DG::fixed + DG::bar_bytes;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int N = m.n_sites, NL = m.n_layers;

    if (tid == 0) {
        // a KV chunk is read by the NSPLIT warps of its sample (each takes its heads): NSPLIT arrivals free a slot;
        // the one warp that consumes a weight chunk arrives NSPLIT times at once
        for (int i = 0; i < NSLOT; ++i) { mbar_init(bar_full + i, 1); mbar_init(bar_empty + i, NSPLIT); }
        *sh_app = 0;
        *sh_issued = 0;
        if (CL) { mbar_init(bar_x, NWC); mbar_init(bar_x + 1, NWC); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();
    const uint32_t crank = CL ? cluster_ctarank() : 0;
    if (CL) cluster_sync_all();                     // the peer's barriers exist before anyone arrives on them
    // work units: a CTA (a cluster in CL mode) walks sample groups; both CTAs of a cluster iterate alike
    const int n_walk = CL ? gridDim.x / 2 : gridDim.x, walk0 = CL ? blockIdx.x / 2 : blockIdx.x;
    const int n_units = CL ? (a.n_groups + 1) / 2 : a.n_groups;

    // =============================== PRODUCER WARP ===============================
    // Lanes work on VW consecutive chunks of the ring at once (one chunk per lane: wait for the
    // slot, arm the mbarrier, one bulk copy per run).  VW <= NSLOT, so a lane only ever waits
    // on a chunk issued in an earlier round -- no circular wait with the consumers.
    if (warp >= NWC) {
        // The KV rows stream through L2 once per step (one step of the whole batch touches more bytes than L2
        // holds, so none of them survives until its next use): read them evict_first so that they do not push out
        // the GEMM weights every CTA re-reads.  cfg5: 265.6 -> 258.6 ms; a kept (evict_last) fraction of the rows
        // or evict_last on the weights adds nothing.
        uint64_t kv_pol = 0;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(kv_pol));
        constexpr int VW = NSLOT >= 32 ? 32 : (NSLOT >= 16 ? 16 : (NSLOT >= 8 ? 8 : (NSLOT >= 4 ? 4 : 2)));
        uint32_t seq = 0;
        int it = 0;
        // Chunks are armed strictly in ring order, but as soon as their slot is free: each round the lanes
        // probe the next VW slots once and the leading run of free ones is issued.  (Waiting for all VW
        // slots would hold back the refill of a slot until VW - 1 later chunks had been consumed as well:
        // two or three exposed HBM round trips per attention phase instead of one.)
        auto ready_prefix = [&](bool active, uint32_t slot, uint32_t par) {
            const bool ok = active && mbar_test(bar_empty + slot, par ^ 1u);
            const unsigned int bm = __ballot_sync(0xffffffffu, ok);
            return bm == 0xffffffffu ? 32 : __ffs(~bm) - 1;  // lanes 0 .. npre-1 are all free
        };
        // one weight matrix = n consecutive CHUNK_BYTES pieces of its packed image, one copy each
        auto issue_weights = [&](const uint4* w, int n, int first = 0, int stride = 1) {
            if constexpr (DG::WG > 1) {                 // groups of WG chunks: one copy, bytes counted on the first slot
                constexpr int WG = DG::WG, GB = WG * DG::CHUNK_BYTES;
                const unsigned char* srcg = reinterpret_cast<const unsigned char*>(w);
                const int ng = n / WG;
                for (int g0 = 0; g0 < ng;) {
                    const int gi = g0 + lane;
                    const uint32_t sq = seq + (uint32_t)(gi * WG);
                    const uint32_t slot = sq % NSLOT, par = (sq / NSLOT) & 1u;
                    bool ok = lane < VW / WG && gi < ng;
#pragma unroll
                    for (int k = 0; k < WG; ++k) ok = ok && mbar_test(bar_empty + slot + k, par ^ 1u);
                    const unsigned int bm = __ballot_sync(0xffffffffu, ok);
                    const int npre = bm == 0xffffffffu ? 32 : __ffs(~bm) - 1;
                    if (lane < npre) {
                        mbar_arrive_expect_tx(bar_full + slot, (uint32_t)GB);
#pragma unroll
                        for (int k = 1; k < WG; ++k) mbar_arrive(bar_full + slot + k);
                        bulk_g2s(ring + (size_t)slot * DG::CHUNK_BYTES, srcg + (size_t)gi * GB, (uint32_t)GB, bar_full + slot);
                    }
                    __syncwarp();
                    g0 += npre;
                    if (lane == 0 && npre) st_release_s32(sh_issued, (int)(seq + (uint32_t)(g0 * WG)));
                }
                seq += (uint32_t)n;
                return;
            }
            const unsigned char* src = reinterpret_cast<const unsigned char*>(w) + (size_t)first * DG::CHUNK_BYTES;
            for (int i0 = 0; i0 < n;) {
                const int i = i0 + lane;
                const uint32_t sq = seq + (uint32_t)i;
                const uint32_t slot = sq % NSLOT, par = (sq / NSLOT) & 1u;
                const int npre = ready_prefix(lane < VW && i < n, slot, par);
                if (lane < npre) {
                    mbar_arrive_expect_tx(bar_full + slot, (uint32_t)DG::CHUNK_BYTES);
                    bulk_g2s(ring + (size_t)slot * DG::CHUNK_BYTES, src + (size_t)i * stride * DG::CHUNK_BYTES,
                             (uint32_t)DG::CHUNK_BYTES, bar_full + slot);
                }
                __syncwarp();
                i0 += npre;
                if (lane == 0 && npre) st_release_s32(sh_issued, (int)(seq + (uint32_t)i0));
            }
            seq += (uint32_t)n;
        };
        for (int wu = walk0; wu < n_units; wu += n_walk, ++it) {
            const int unit = CL ? wu * 2 + (int)crank : wu;
            const int b_first = unit < a.n_groups ? unit * a.rows_per_group : 0;
            const int n_own = unit < a.n_groups ? min(a.rows_per_group, a.B - b_first) : 0;   // 0: FFN helper only
            const uint32_t inv_own = n_own > 0 ? (65536u + (uint32_t)n_own - 1u) / (uint32_t)n_own : 0u;
            // copy plan of a step: chunk -> run list (staged in shared memory when it fits)
            struct Plan { int nch, nn, nruns; const int32_t* cptr; const int2* rptr; };
            auto stage_plan = [&](int t) {
                Plan p;
                if (t >= N) { p.nch = p.nn = p.nruns = 0; p.cptr = nullptr; p.rptr = nullptr; return p; }
                const int cp0 = __ldg(m.d_chunk_ptr + t);
                p.nch = __ldg(m.d_chunk_ptr + t + 1) - cp0;
                p.nn = __ldg(m.d_nn + t);
                const int rp0 = __ldg(m.d_chunk_run_ptr + cp0);
                p.nruns = __ldg(m.d_chunk_run_ptr + cp0 + p.nch) - rp0;
                int32_t* tc = tab_c + (t & 1) * DG::TAB_C;
                int2* tr = tab_r + (t & 1) * DG::TAB_R;
                __syncwarp();
                if (p.nch + 1 <= DG::TAB_C && p.nruns <= DG::TAB_R) {
                    for (int i = lane; i <= p.nch; i += 32) tc[i] = __ldg(m.d_chunk_run_ptr + cp0 + i) - rp0;
                    for (int i = lane; i < p.nruns; i += 32) tr[i] = __ldg(m.d_runs + rp0 + i);
                    __syncwarp();
                    p.cptr = tc; p.rptr = tr;
                } else {
                    p.cptr = m.d_chunk_run_ptr + cp0; p.rptr = m.d_runs;      // absolute run indices
                }
                return p;
            };
            Plan cur = stage_plan(0);
            for (int t = 0; t < N; ++t) {
                const Plan nxt = stage_plan(t + 1);
                const int nch = cur.nch, nn = cur.nn;
                const int32_t* cptr = cur.cptr;
                const int2* rptr = cur.rptr;
                const int total = n_own * nch;
                for (int l = 0; l < NL; ++l) {
                    const FvLayerDev& L = m.layer[l];
                    if (DG::WRING) issue_weights(L.wqkv, DG::NQ);
                    if (total > 0) {
                        // rows < t of layer l are complete once step t-1 has appended at layer l
                        const int need = (it * N + (t - 1)) * NL + l + 1;
                        while (ld_acquire_s32(sh_app) < need) __nanosleep(32);
                    }
                    const unsigned char* src_l = reinterpret_cast<const unsigned char*>(
                        m.kv_s + ((size_t)b_first * NL + l) * m.kv_rows * (2 * D));
                    for (int i0 = 0; i0 < total;) {
                        const int i = i0 + lane;
                        const uint32_t sq = seq + (uint32_t)i;
                        const uint32_t slot = sq % NSLOT, par = (sq / NSLOT) & 1u;
                        const int npre = ready_prefix(lane < VW && i < total, slot, par);
                        if (lane < npre) {
                            // chunk-major inside a round of GR samples (= the samples the compute
                            // warps work on at the same time), rounds in order: every warp then
                            // consumes its chunks in ring order
                            // (one round when all rows are attended at once; then c = i / n_own by multiply and shift,
                            // exact below 2048 for divisors up to 32 -- two integer divisions were a fifth of a round)
                            int k = 0, rem = i;
                            if constexpr (R > GR) { k = i / (GR * nch); rem = i - k * GR * nch; }
                            const int nk = R > GR ? min(GR, n_own - k * GR) : n_own;
                            const int c = (R <= GR && total < 2048) ? (int)(((uint32_t)rem * inv_own) >> 16) : rem / nk;
                            const int r = k * GR + (rem - c * nk);
                            const int rows = min(CH, nn - c * CH);
                            mbar_arrive_expect_tx(bar_full + slot, (uint32_t)rows * DG::ROW_BYTES);
                            const unsigned char* src = src_l + (size_t)r * NL * m.kv_rows * DG::ROW_BYTES;
                            unsigned char* dst = ring + (size_t)slot * DG::CHUNK_BYTES;
                            const int j1 = cptr[c + 1];
                            for (int j = cptr[c]; j < j1; ++j) {
                                const int2 run = rptr[j];
                                bulk_g2s_hint(dst + (size_t)(run.y >> 16) * DG::ROW_BYTES, src + (size_t)run.x * DG::ROW_BYTES,
                                              (uint32_t)(run.y & 0xffff) * DG::ROW_BYTES, bar_full + slot, kv_pol);
                            }
                        }
                        __syncwarp();
                        i0 += npre;
                        if (lane == 0 && npre) st_release_s32(sh_issued, (int)(seq + (uint32_t)i0));
                    }
                    seq += (uint32_t)total;
                    if constexpr (DG::WG > 1) {           // empty chunks up to the next multiple of WG: armed and released here
                        const int pad = (DG::WG - total % DG::WG) % DG::WG;
                        if (lane == 0)
                            for (int k = 0; k < pad; ++k) {
                                const uint32_t sq = seq + (uint32_t)k;
                                const uint32_t slot = sq % NSLOT, par = (sq / NSLOT) & 1u;
                                while (!mbar_test(bar_empty + slot, par ^ 1u)) {}
                                mbar_arrive(bar_full + slot);
                                mbar_arrive_n(bar_empty + slot, NSPLIT);
                            }
                        __syncwarp();
                        seq += (uint32_t)pad;
                        if (lane == 0 && pad) st_release_s32(sh_issued, (int)seq);
                    }
                    if (DG::WRING) {
                        if (m.has_wo) issue_weights(L.wo, DG::NO);
                        if (CL) {     // my half of the hidden layer: rows of W1, K-half of every m-tile of W2
                            issue_weights(L.w1, DG::N1 / 2, (int)crank * (DG::N1 / 2));
                            issue_weights(L.w2, DG::N2 / 2, (int)crank, 2);
                        } else {
                            issue_weights(L.w1, DG::N1);
                            issue_weights(L.w2, DG::N2);
                        }
                    }
                }
                cur = nxt;
            }
        }
        if (CL) cluster_sync_all();                 // matches the compute warps' final cluster barrier
        return;
    }

    // =============================== COMPUTE WARPS ===============================
    const int g = lane >> 2, c4 = lane & 3;
    const int rg = lane / LPR, sub = lane % LPR;
    uint32_t seq_base = 0;
    int it = 0;
    const RingCtx rc{ring, bar_full, bar_empty, sh_issued};
    // sh_par holds: [0, PAR_E) ln1_g | ln1_b | bqkv of the layer about to run (loaded during the attention phase of the
    // layer before it), [PAR_E, PAR_E + PAR_L) ln2_g | ln2_b | b1 | b2 | bo of the running layer (loaded during its LN1
    // phase); thread pidx takes float4 number pidx, highest warps first (they have the least other work)
    const int pidx = NWC * 32 - 1 - tid;
    if (pidx < DG::PAR_E / 4)
        reinterpret_cast<float4*>(sh_par)[pidx] = __ldg(reinterpret_cast<const float4*>(m.layer[0].par) + pidx);
    for (int wu = walk0; wu < n_units; wu += n_walk, ++it) {
        const int unit = CL ? wu * 2 + (int)crank : wu;
        const int b_first = unit < a.n_groups ? unit * a.rows_per_group : 0;
        const int n_own = unit < a.n_groups ? min(a.rows_per_group, a.B - b_first) : 0;       // 0: FFN helper only
        if (tid < R) { sh_tok[tid] = 0; sh_logq[tid] = 0.0; }
        for (int t = 0; t < N; ++t) {
            const int me0 = __ldg(m.mask_rowptr + t);
            const int nn = __ldg(m.d_nn + t);                        // rows that come through the ring
            const int nch = (nn + CH - 1) / CH;
            int dir_pos[FV_DIRECT_MAX];                              // isolated key positions, loaded straight from the pool
#pragma unroll
            for (int i = 0; i < FV_DIRECT_MAX; ++i) dir_pos[i] = __ldg(m.d_dir + (size_t)t * FV_DIRECT_MAX + i);
            if (tid < R) sh_u[tid] = tid < n_own ? __ldg(a.uniforms + (size_t)(b_first + tid) * N + t) : 2.f;
            cbar();
            // ---- concatenated positional embedding (Eq. 15, l.287-292) -------------------
            for (int i = tid; i < R * D; i += NWC * 32) {
                const int r = i / D, f = i - r * D;
                const int dt = m.d_token;
                sh_h[r * HS + f] = f < dt ? __ldg(m.tok_emb + sh_tok[r] * dt + f)
                                          : __ldg(m.posemb + (size_t)t * (D - dt) + (f - dt));
            }
            cbar();
            for (int l = 0; l < NL; ++l) {
                const FvLayerDev& L = m.layer[l];
                // ---- LN1 (Alg. 2 l.12) -> bf16 activations ----------------------------------
                float4 pl = make_float4(0.f, 0.f, 0.f, 0.f);
                if (pidx < DG::PAR_L / 4) pl = __ldg(reinterpret_cast<const float4*>(L.par + DG::PAR_E) + pidx);
                for (int r = warp; r < R; r += NWC)
                    ln_row<D, true>(sh_h + r * HS, sh_par, sh_par + D, m.ln_eps, false, sh_a + r * AS, lane);
                if (pidx < DG::PAR_L / 4) reinterpret_cast<float4*>(sh_par + DG::PAR_E)[pidx] = pl;
                cbar();
                // ---- q, k, v = W a + b (Eq. 2; Alg. 2 l.13) ---------------------------------
                {
                    auto epi = [&](int mt, int, float (&acc)[NT][4]) {
                        const int f = mt * 16 + g;
                        const float b0 = sh_par[2 * D + f], b1 = sh_par[2 * D + f + 8];
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) {
                            const int row = nt * 8 + 2 * c4;
                            if (f < D) {                         // whole m-tile is q (warp-uniform)
                                float* o = sh_q + row * QS2 + f;
                                o[0] = acc[nt][0] + b0; o[QS2] = acc[nt][1] + b0;
                                o[8] = acc[nt][2] + b1; o[QS2 + 8] = acc[nt][3] + b1;
                            } else {
                                __nv_bfloat16* o = sh_kv + row * KVS + (f - D);
                                o[0] = __float2bfloat16_rn(acc[nt][0] + b0); o[KVS] = __float2bfloat16_rn(acc[nt][1] + b0);
                                o[8] = __float2bfloat16_rn(acc[nt][2] + b1); o[KVS + 8] = __float2bfloat16_rn(acc[nt][3] + b1);
                            }
                        }
                    };
                    if constexpr (DG::WRING) {
                        gemm_ring<D / 16, NT, DG::TPCH, NSLOT, DG::CHUNK_BYTES, DG::WG, NSPLIT>(rc, DG::NQ, seq_base, sh_a, AS, warp, lane, epi);
                        seq_base += DG::NQ;
                    } else {
                        gemm_rows<D / 16, 1, NT, NWC, GEMM_MAXL>(L.wqkv, 3 * D / 16, sh_a, AS, warp, lane, epi);
                    }
                }
                cbar();
                // ---- append k_t, v_t to the KV pool as bf16 (Alg. 2 l.17; reading A2) -------
                // The warps without an attention task (sample slots the CTA does not own: 2 of 16 warps at 7 samples) take
                // the whole append and its proxy fence off the others' path to their first KV chunk; with every slot owned
                // all threads share it.  The producer reads these rows through the async proxy (cp.async.bulk); they are
                // first needed one step later, so the append shares its barrier with the attention phase and is
                // published after it.
                {
                    const int busy = n_own * NSPLIT < NWC ? n_own * NSPLIT : 0;       // warps below `busy` skip the append
                    if (warp >= busy) {
                        for (int i = tid - busy * 32; i < R * (2 * D / 8); i += (NWC - busy) * 32) {
                            const int r = i / (2 * D / 8), ch = i - r * (2 * D / 8);
                            if (r >= n_own) continue;
                            const uint4 v = *reinterpret_cast<const uint4*>(sh_kv + r * KVS + ch * 8);
                            __nv_bfloat16* dst = m.kv_s + (((size_t)(b_first + r) * NL + l) * m.kv_rows + t % m.kv_rows) * (2 * D) + ch * 8;
                            *reinterpret_cast<uint4*>(dst) = v;
                        }
                        asm volatile("fence.proxy.async.global;\n" ::: "memory");
                    }
                }
                float4 pe = make_float4(0.f, 0.f, 0.f, 0.f);
                if (pidx < DG::PAR_E / 4) pe = __ldg(reinterpret_cast<const float4*>(m.layer[l + 1 < NL ? l + 1 : 0].par) + pidx);
                // ---- masked attention from the KV ring + residual (Eq. 3; Alg. 2 l.14-15) ---
                // The NSPLIT warps of a sample split the query row by HEADS: warp (r, sp) scores all rows of A(t) against
                // its D / NSPLIT features and owns the finished output of those heads -- no partial results to merge
                // between warps, no extra phase; both read every KV chunk of the sample (slots count NSPLIT arrivals).
                for (int task = warp; task < R * NSPLIT; task += NWC) {
                    const int r = task / NSPLIT, sp = task - r * NSPLIT;
                    if (r >= n_own) continue;
                    constexpr int DS = D / NSPLIT, LPRS = DS / 8;          // features / lanes of a warp's part of a row
                    const int rgs = lane / LPRS, subs = lane - rgs * LPRS;
                    const float qs = kLog2e * rsqrtf((float)DH);
                    const float* qrow = sh_q + r * QS2 + sp * DS;
                    const __nv_bfloat16* kvrow = sh_kv + r * KVS + sp * DS;
                    float q[8], acc[8];
                    {                                    // (rows are 16-byte aligned: QS2, KVS and the offsets are multiples of 16 B)
                        const float4 qa = *reinterpret_cast<const float4*>(qrow + subs * 8), qb = *reinterpret_cast<const float4*>(qrow + subs * 8 + 4);
                        q[0] = qa.x * qs; q[1] = qa.y * qs; q[2] = qa.z * qs; q[3] = qa.w * qs;
                        q[4] = qb.x * qs; q[5] = qb.y * qs; q[6] = qb.z * qs; q[7] = qb.w * qs;
                    }
                    float mm = -1e30f, ll = 0.f;
#pragma unroll
                    for (int j = 0; j < 8; ++j) acc[j] = 0.f;
                    {                                    // row t itself, as the pool stores it (bf16)
                        const uint4 ks = *reinterpret_cast<const uint4*>(kvrow + subs * 8), vs = *reinterpret_cast<const uint4*>(kvrow + D + subs * 8);
                        const uint32_t kw[4] = {ks.x, ks.y, ks.z, ks.w}, vw[4] = {vs.x, vs.y, vs.z, vs.w};
                        float d = 0.f;
#pragma unroll
                        for (int j = 0; j < 4; ++j) { d += q[2 * j] * bf_lo(kw[j]); d += q[2 * j + 1] * bf_hi(kw[j]); }
#pragma unroll
                        for (int o = 1; o < LPH; o <<= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
                        if (rgs == 0) {
                            mm = d; ll = 1.f;
#pragma unroll
                            for (int j = 0; j < 4; ++j) { acc[2 * j] = bf_lo(vw[j]); acc[2 * j + 1] = bf_hi(vw[j]); }
                        }
                    }
                    // The step's isolated rows, RPID per load: row group g takes row b0 + g.  The first set is requested now and
                    // used after the ring's rows; further sets (lattice edges, 3D masks) are loaded then.  (Rows this CTA wrote
                    // in an earlier step with plain stores; barriers since.)
                    constexpr int RPID = 32 / LPRS;
                    auto dir_load = [&](int b0, uint4& k4, uint4& v4) {
                        int dpos = -1;
#pragma unroll
                        for (int i = 0; i < RPID; ++i) if (rgs == i && b0 + i < FV_DIRECT_MAX) dpos = dir_pos[b0 + i < FV_DIRECT_MAX ? b0 + i : 0];
                        k4 = v4 = make_uint4(0u, 0u, 0u, 0u);
                        if (dpos >= 0) {
                            const __nv_bfloat16* dp = m.kv_s + (((size_t)(b_first + r) * NL + l) * m.kv_rows + dpos) * (2 * D) + sp * DS + subs * 8;
                            k4 = *reinterpret_cast<const uint4*>(dp);
                            v4 = *reinterpret_cast<const uint4*>(dp + D);
                        }
                        return dpos >= 0;
                    };
                    uint4 dk, dv;
                    const bool dok = dir_load(0, dk, dv);
                    for (int c = 0; c < nch; ++c) {
                        const int kr = r / GR, nk = min(GR, n_own - kr * GR);
                        const uint32_t sq = seq_base + (uint32_t)(kr * GR * nch + c * nk + (r - kr * GR));
                        uint32_t slot;
                        const unsigned char* chunk = ring_acquire<NSLOT, DG::CHUNK_BYTES>(rc, sq, slot);
                        attend_chunk<D, DH, CH, NSPLIT>(chunk + sp * DS * 2, min(CH, nn - c * CH), q, rgs, subs, mm, ll, acc);
                        // every K word fed the scores behind ll, V words x / y / z / w fed acc[0..1] / [2..3] / [4..5] / [6..7]
                        ring_release_dep(rc, slot, lane, 1, __float_as_uint(ll) ^ __float_as_uint(acc[0]) ^ __float_as_uint(acc[2]) ^
                                                                __float_as_uint(acc[4]) ^ __float_as_uint(acc[6]));
                    }
                    if (dir_pos[0] >= 0) attend_direct<DH>(dk, dv, dok, q, mm, ll, acc);
#pragma unroll
                    for (int b0 = RPID; b0 < FV_DIRECT_MAX; b0 += RPID) {
                        if (dir_pos[b0] < 0) break;
                        uint4 k4, v4;
                        const bool ok4 = dir_load(b0, k4, v4);
                        attend_direct<DH>(k4, v4, ok4, q, mm, ll, acc);
                    }
#pragma unroll
                    for (int o = LPRS; o < 32; o <<= 1) {      // merge the row groups of the warp
                        const float m2 = __shfl_xor_sync(0xffffffffu, mm, o);
                        const float l2 = __shfl_xor_sync(0xffffffffu, ll, o);
                        const float mx = fmaxf(mm, m2);
                        const float c1 = fast_exp2(mm - mx), c2 = fast_exp2(m2 - mx);
                        ll = ll * c1 + l2 * c2;
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const float a2 = __shfl_xor_sync(0xffffffffu, acc[j], o);
                            acc[j] = acc[j] * c1 + a2 * c2;
                        }
                        mm = mx;
                    }
                    if (lane < LPRS) {
                        const float inv = 1.0f / ll;
                        if (m.has_wo) {
#pragma unroll
                            for (int j = 0; j < 8; ++j) sh_a[r * AS + sp * DS + lane * 8 + j] = __float2bfloat16_rn(acc[j] * inv);
                        } else {
#pragma unroll
                            for (int j = 0; j < 8; ++j) sh_h[r * HS + sp * DS + lane * 8 + j] += acc[j] * inv;
                        }
                    }
                }
                seq_base += (uint32_t)(n_own * nch);
                if constexpr (DG::WG > 1) seq_base += (uint32_t)((DG::WG - (n_own * nch) % DG::WG) % DG::WG);
                if (pidx < DG::PAR_E / 4) reinterpret_cast<float4*>(sh_par)[pidx] = pe;
                cbar();
                if (tid == 0) st_release_s32(sh_app, (it * N + t) * NL + l + 1);
                // ---- optional output projection (bypassed in the paper, l.107) --------------
                if (m.has_wo) {
                    {
                    auto epi = [&](int mt, int, float (&acc)[NT][4]) {
                            const int f = mt * 16 + g;
                            const float b0 = sh_par[12 * D + f], b1 = sh_par[12 * D + f + 8];
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt) {
                                float* o = sh_h + (nt * 8 + 2 * c4) * HS + f;
                                o[0] += acc[nt][0] + b0; o[HS] += acc[nt][1] + b0;
                                o[8] += acc[nt][2] + b1; o[HS + 8] += acc[nt][3] + b1;
                            }
                        };
                    if constexpr (DG::WRING) {
                        gemm_ring<D / 16, NT, DG::TPCH, NSLOT, DG::CHUNK_BYTES, DG::WG, NSPLIT>(rc, DG::NO, seq_base, sh_a, AS, warp, lane, epi);
                        seq_base += DG::NO;
                    } else {
                        gemm_rows<D / 16, 1, NT, NWC, GEMM_MAXL>(L.wo, D / 16, sh_a, AS, warp, lane, epi);
                    }
                }
                    cbar();
                }
                if constexpr (CL) {
                    // ======== FFN split over the 2-CTA cluster =====================================
                    // Each CTA streams only HALF of W1/W2 (its 2D hidden columns) and applies them to
                    // the rows of BOTH CTAs; the halves meet again as two partial sums.
                    const uint32_t peer = crank ^ 1u;
                    const uint32_t xpar = (uint32_t)((((long long)it * N + t) * NL + l) & 1);
                    // ---- LN2 of my rows -> my slot of sh_a2, copy to the peer's sh_a2 -------------
                    for (int r = warp; r < R; r += NWC)
                        ln_row<D, true>(sh_h + r * HS, sh_par + 5 * D, sh_par + 6 * D, m.ln_eps, m.ln2_style == 1,
                                        sh_a2 + (crank * R + r) * AS, lane);
                    cbar();
                    {
                        constexpr int PCS = R * AS * 2 / 16;            // 16-byte pieces of my R rows
                        const unsigned char* src = reinterpret_cast<const unsigned char*>(sh_a2 + crank * R * AS);
                        const uint32_t dst = map_to_peer(smem_u32(src), peer);
                        for (int i = tid; i < PCS; i += NWC * 32)
                            st_peer128(dst + i * 16, *reinterpret_cast<const uint4*>(src + i * 16));
                        __syncwarp();
                        if (lane == 0) mbar_arrive_peer(map_to_peer(smem_u32(bar_x), peer));
                    }
                    mbar_wait_cluster(bar_x, xpar);
                    // ---- FFN1 half + GELU over 2R rows -> bf16 hidden half ------------------------
                    {
                        auto epi = [&](int mt, int, float (&acc)[NT2][4]) {
                            const int f = mt * 16 + g;
                            const float b0 = sh_par[7 * D + crank * 2 * D + f], b1 = sh_par[7 * D + crank * 2 * D + f + 8];
#pragma unroll
                            for (int nt = 0; nt < NT2; ++nt) {
                                __nv_bfloat16* o = sh_hid + (nt * 8 + 2 * c4) * FS2 + f;
                                // exact-erf GELU by the one-ex2 erfc form (fv_device.cuh; erff cost a tenth of the kernel's issue slots)
                                const uint32_t g0 = gelu_erfc_x2(acc[nt][0] + b0, acc[nt][1] + b0);
                                const uint32_t g1 = gelu_erfc_x2(acc[nt][2] + b1, acc[nt][3] + b1);
                                uint16_t* ou = reinterpret_cast<uint16_t*>(o);
                                ou[0] = (uint16_t)g0; ou[FS2] = (uint16_t)(g0 >> 16);
                                ou[8] = (uint16_t)g1; ou[FS2 + 8] = (uint16_t)(g1 >> 16);
                            }
                        };
                        gemm_ring<D / 16, NT2, DG::TPCH, NSLOT, DG::CHUNK_BYTES, DG::WG, NSPLIT>(rc, DG::N1 / 2, seq_base, sh_a2, AS, warp, lane, epi);
                        seq_base += DG::N1 / 2;
                    }
                    cbar();
                    // ---- FFN2 over my K-half: partial sums for all 2R rows -------------------------
                    {
                        auto epi = [&](int mt, int, float (&acc)[NT2][4]) {
                            const int f = mt * 16 + g;
#pragma unroll
                            for (int nt = 0; nt < NT2; ++nt) {
                                float* o = sh_part + (nt * 8 + 2 * c4) * HS + f;
                                o[0] = acc[nt][0]; o[HS] = acc[nt][1];
                                o[8] = acc[nt][2]; o[HS + 8] = acc[nt][3];
                            }
                        };
                        gemm_ring<2 * D / 16, NT2, DG::TPCH, NSLOT, DG::CHUNK_BYTES, DG::WG, NSPLIT>(rc, DG::N2 / 2, seq_base, sh_hid, FS2, warp, lane, epi);
                        seq_base += DG::N2 / 2;
                    }
                    cbar();
                    {   // the peer's rows of my partial sums -> the peer's sh_xp
                        constexpr int PCS = R * HS * 4 / 16;
                        const unsigned char* src = reinterpret_cast<const unsigned char*>(sh_part + peer * R * HS);
                        const uint32_t dst = map_to_peer(smem_u32(sh_xp), peer);
                        for (int i = tid; i < PCS; i += NWC * 32)
                            st_peer128(dst + i * 16, *reinterpret_cast<const uint4*>(src + i * 16));
                        __syncwarp();
                        if (lane == 0) mbar_arrive_peer(map_to_peer(smem_u32(bar_x + 1), peer));
                    }
                    mbar_wait_cluster(bar_x + 1, xpar);
                    // ---- feed-forward residual; the two halves are added in cluster-rank order ----
                    for (int i = tid; i < R * D; i += NWC * 32) {
                        const int r = i / D, f = i - r * D;
                        const float mine = sh_part[(crank * R + r) * HS + f], theirs = sh_xp[r * HS + f];
                        const float p0 = crank == 0 ? mine : theirs, p1 = crank == 0 ? theirs : mine;
                        sh_h[r * HS + f] += (p0 + p1) + sh_par[11 * D + f];
                    }
                    cbar();
                } else {
                    // ---- LN2 (Alg. 2 l.16; ln2_style 1 = Alg. 1 l.5) ----------------------------
                    for (int r = warp; r < R; r += NWC)
                        ln_row<D, true>(sh_h + r * HS, sh_par + 5 * D, sh_par + 6 * D, m.ln_eps, m.ln2_style == 1, sh_a + r * AS, lane);
                    cbar();
                    // ---- FFN up-projection + exact GELU -> bf16 hidden ---------------------------
                    {
                        auto epi = [&](int mt, int, float (&acc)[NT][4]) {
                            const int f = mt * 16 + g;
                            const float b0 = sh_par[7 * D + f], b1 = sh_par[7 * D + f + 8];
    #pragma unroll
                            for (int nt = 0; nt < NT; ++nt) {
                                __nv_bfloat16* o = sh_hid + (nt * 8 + 2 * c4) * FS + f;
                                // exact-erf GELU by the one-ex2 erfc form (fv_device.cuh; erff cost a tenth of the kernel's issue slots)
                                const uint32_t g0 = gelu_erfc_x2(acc[nt][0] + b0, acc[nt][1] + b0);
                                const uint32_t g1 = gelu_erfc_x2(acc[nt][2] + b1, acc[nt][3] + b1);
                                uint16_t* ou = reinterpret_cast<uint16_t*>(o);
                                ou[0] = (uint16_t)g0; ou[FS] = (uint16_t)(g0 >> 16);
                                ou[8] = (uint16_t)g1; ou[FS + 8] = (uint16_t)(g1 >> 16);
                            }
                        };
                        if constexpr (DG::WRING) {
                            gemm_ring<D / 16, NT, DG::TPCH, NSLOT, DG::CHUNK_BYTES, DG::WG, NSPLIT>(rc, DG::N1, seq_base, sh_a, AS, warp, lane, epi);
                            seq_base += DG::N1;
                        } else {
                            gemm_rows<D / 16, 1, NT, NWC, GEMM_MAXL>(L.w1, 4 * D / 16, sh_a, AS, warp, lane, epi);
                        }
                    }
                    cbar();
                    // ---- FFN down-projection + residual (Alg. 2 l.16) ---------------------------------
                    if constexpr (DG::NO_PART) {
                        // a warp takes whole m-tiles (both K-halves from consecutive ring chunks): the
                        // accumulator goes straight into the residual stream
                        auto epi = [&](int mt, float (&acc)[NT][4]) {
                            const int f = mt * 16 + g;
                            const float b0 = sh_par[11 * D + f], b1 = sh_par[11 * D + f + 8];
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt) {
                                float* o = sh_h + (nt * 8 + 2 * c4) * HS + f;
                                o[0] += acc[nt][0] + b0; o[HS] += acc[nt][1] + b0;
                                o[8] += acc[nt][2] + b1; o[HS + 8] += acc[nt][3] + b1;
                            }
                        };
                        gemm_ring_kparts<4 * D / 16, NT, DG::TPCH, NSLOT, DG::CHUNK_BYTES, DG::WG, NSPLIT>(rc, D / 16, seq_base, sh_hid, FS, warp, lane, epi);
                        seq_base += DG::N2;
                        cbar();
                    } else {
                        auto epi = [&](int mt, int ks, float (&acc)[NT][4]) {
                            const int f = mt * 16 + g;
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt) {
                                float* o = sh_part + ((size_t)ks * R + nt * 8 + 2 * c4) * HS + f;
                                o[0] = acc[nt][0]; o[HS] = acc[nt][1];
                                o[8] = acc[nt][2]; o[HS + 8] = acc[nt][3];
                            }
                        };
                        if constexpr (DG::WRING) {
                            gemm_ring<4 * D / 16, NT, DG::TPCH, NSLOT, DG::CHUNK_BYTES, DG::WG, NSPLIT>(rc, DG::N2, seq_base, sh_hid, FS, warp, lane, epi);
                            seq_base += DG::N2;
                        } else {
                            gemm_rows<4 * D / 16, KS2, NT, NWC, GEMM_MAXL>(L.w2, D / 16, sh_hid, FS, warp, lane, epi);
                        }
                        cbar();
                        for (int i = tid; i < R * D; i += NWC * 32) {
                            const int r = i / D, f = i - r * D;
                            float v = sh_par[11 * D + f];
#pragma unroll
                            for (int ks = 0; ks < KS2; ++ks) v += sh_part[((size_t)ks * R + r) * HS + f];
                            sh_h[r * HS + f] += v;
                        }
                        cbar();
                    }

                }
            }
            // ---- patch tokens (SI I.D, l.603-605): V-way softmax head, token = first k with u < p_0 + .. + p_k ----
            if (m.vocab > 2) {
                const int V = m.vocab;
                for (int r = warp; r < R; r += NWC) {
                    if (r >= n_own) continue;
                    const int b = b_first + r;
                    // lane owns tokens lane, lane + 32, ...: logits, then everything in token order
                    float z[8];
                    float mx = -INFINITY;
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int k = lane + 32 * i;
                        z[i] = -INFINITY;
                        if (k < V) {
                            const float4* wr = reinterpret_cast<const float4*>(m.head_w + (size_t)k * D);
                            float acc = __ldg(m.head_b + k);
#pragma unroll 4
                            for (int f4 = 0; f4 < D / 4; ++f4) {
                                const float4 wv = __ldg(wr + f4);
                                const float4 hv = *reinterpret_cast<const float4*>(sh_h + r * HS + f4 * 4);
                                acc += hv.x * wv.x + hv.y * wv.y + hv.z * wv.z + hv.w * wv.w;
                            }
                            z[i] = acc;
                            mx = fmaxf(mx, acc);
                        }
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
                    float e[8], mine = 0.f;
#pragma unroll
                    for (int i = 0; i < 8; ++i) { e[i] = lane + 32 * i < V ? expf(z[i] - mx) : 0.f; mine += e[i]; }
                    const float S = warp_sum(mine);
                    // running sums in token order: block i (tokens 32 i .. 32 i + 31) after the blocks before it
                    const float target = sh_u[r] * S;               // u < cdf_k  <=>  u S < e_0 + .. + e_k
                    float carry = 0.f;
                    int tok = V - 1;
                    bool found = false;
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        if (32 * i >= V) break;
                        float pre = e[i];                            // inclusive scan over the lanes
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) {
                            const float up = __shfl_up_sync(0xffffffffu, pre, o);
                            if (lane >= o) pre += up;
                        }
                        pre += carry;
                        const unsigned hit = __ballot_sync(0xffffffffu, lane + 32 * i < V && target < pre);
                        if (!found && hit) { tok = 32 * i + __ffs(hit) - 1; found = true; }
                        carry = __shfl_sync(0xffffffffu, pre, 31);
                    }
                    // the drawn token's logit and weight live in lane tok % 32, slot tok / 32
                    float zt = 0.f, et = 0.f;
#pragma unroll
                    for (int i = 0; i < 8; ++i) if (i == (tok >> 5)) { zt = z[i]; et = e[i]; }
                    zt = __shfl_sync(0xffffffffu, zt, tok & 31);
                    et = __shfl_sync(0xffffffffu, et, tok & 31);
                    if (lane == 0) {
                        a.spins_out[(size_t)b * N + t] = (int8_t)(uint8_t)tok;
                        sh_tok[r] = tok;
                        sh_logp[r] = (zt - mx) - logf(S);
                        if (a.cond_p) a.cond_p[(size_t)b * N + t] = et / S;
                    }
                }
            } else
            // ---- output head: p(+1) = softmax(z)[1] = sigmoid(z1 - z0) (Alg. 2 l.20-22) -----
            for (int r = warp; r < R; r += NWC) {
                if (r >= n_own) continue;
                const int b = b_first + r;
                float d = 0.f;
#pragma unroll
                for (int j = 0; j < D / 32; ++j) d += sh_h[r * HS + lane * (D / 32) + j] * __ldg(m.head_wd + lane * (D / 32) + j);
                d = warp_sum(d) + m.head_bd;
                if (lane == 0) {
                    const float p = 1.0f / (1.0f + expf(-d));
                    const int up = sh_u[r] < p;                            // reading A10 (l.23)
                    a.spins_out[(size_t)b * N + t] = up ? 1 : -1;           // sigma = 2 s - 1 (l.25)
                    sh_tok[r] = up;
                    const float x = up ? -d : d;                           // log p(s) = -softplus(x)
                    sh_logp[r] = -(fmaxf(x, 0.f) + log1pf(expf(-fabsf(x))));
                    if (a.cond_p) a.cond_p[(size_t)b * N + t] = p;
                }
            }
            cbar();
            // ---- log q accumulation in fp64, fixed order (Alg. 1 l.9) --------------------------
            if (tid < n_own) {
                sh_logq[tid] += (double)sh_logp[tid];
                if (t == N - 1) a.logq[b_first + tid] = (float)sh_logq[tid];
            }
        }
        cbar();
    }
    if (CL) cluster_sync_all();                     // no CTA leaves while its peer may still write to it
}

}  // namespace

// ------------------------------------------------------------------------------ dispatch
template <int D, int DH, int NT, bool CL>
static cudaError_t launch_dec(const FvModelDev& m, const FvForwardArgs& a, int n_sms, cudaStream_t s) {
    auto kern = fv_decode_kernel<D, DH, NT, CL>;
    using DG = DecGeo<D, NT, CL>;
    const size_t smem = DG::total;
    if (cudaError_t e = fv_smem_attr((const void*)kern, (int)DG::total); e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg{};
    cfg.blockDim = dim3(NTHREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    if (CL) {                                     // one CTA per SM, paired: cluster k walks group pairs k, k + n, ...
        const int pairs = (a.n_groups + 1) / 2, max_pairs = n_sms / 2;
        cfg.gridDim = dim3(2 * (pairs < max_pairs ? pairs : max_pairs));
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
    } else {
        cfg.gridDim = dim3(a.n_groups < n_sms ? a.n_groups : n_sms);
    }
    return cudaLaunchKernelEx(&cfg, kern, m, a);
}

template <int D, int DH, bool CL>
static cudaError_t launch_dec_nt(const FvModelDev& m, int nt, const FvForwardArgs& a, int n_sms, cudaStream_t s) {
    switch (nt) {
        case 1: return launch_dec<D, DH, 1, CL>(m, a, n_sms, s);
        case 2: return launch_dec<D, DH, 2, CL>(m, a, n_sms, s);
        case 4: return launch_dec<D, DH, 4, CL>(m, a, n_sms, s);
        default: return cudaErrorInvalidValue;
    }
}

// cluster = 1: 2-CTA clusters split the FFN (needs the weight ring: d <= 128, and no W_O variant yet).
cudaError_t fv_launch_decode(const FvModelDev& m, int d_model, int d_head, int nt, const FvForwardArgs& a,
                             int n_sms, int cluster, cudaStream_t s) {
    const int key = d_model * 1000 + d_head;
    if (cluster && d_model <= 128) {
        switch (key) {
            case 32016: return launch_dec_nt<32, 16, true>(m, nt, a, n_sms, s);
            case 64016: return launch_dec_nt<64, 16, true>(m, nt, a, n_sms, s);
            case 64032: return launch_dec_nt<64, 32, true>(m, nt, a, n_sms, s);
            case 128032: return launch_dec_nt<128, 32, true>(m, nt, a, n_sms, s);
            case 128016: return launch_dec_nt<128, 16, true>(m, nt, a, n_sms, s);
            default: break;
        }
    }
    switch (key) {
        case 32016: return launch_dec_nt<32, 16, false>(m, nt, a, n_sms, s);
        case 64016: return launch_dec_nt<64, 16, false>(m, nt, a, n_sms, s);
        case 64032: return launch_dec_nt<64, 32, false>(m, nt, a, n_sms, s);
        case 128032: return launch_dec_nt<128, 32, false>(m, nt, a, n_sms, s);
        case 256064: return launch_dec_nt<256, 64, false>(m, nt, a, n_sms, s);
        case 128016: return launch_dec_nt<128, 16, false>(m, nt, a, n_sms, s);
        default: return cudaErrorInvalidValue;
    }
}
