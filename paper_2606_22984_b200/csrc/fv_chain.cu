// fv_chain.cu -- weight-stationary sampler of fv_sample (Alg. 2) for sm_100a, d = 128.
//
// A thread-block CLUSTER of n_layers CTAs is a pipeline: CTA l keeps ALL weights of layer l on chip for
// the whole launch -- W_qkv and W_1 in TENSOR MEMORY (448 of the 512 columns, as the A operand of
// tcgen05.mma), W_2 in shared memory (128 KB, SWIZZLE_128B image) -- so no GEMM weight is ever streamed
// again (fv_decode.cu re-reads 360 KB per CTA and layer-step).  Micro-batches of R <= 16 samples travel
// down the chain: CTA l runs layer l of Alg. 2 for the micro-batch (LN1 -> QKV -> KV append -> masked
// attention from its own KV ring -> LN2 -> FFN -> residual) and hands the residual stream (R x 512 B)
// to CTA l + 1 through DISTRIBUTED SHARED MEMORY; the last CTA applies the head, draws the spin from the
// caller's uniform, accumulates log q and sends the token back to CTA 0, which embeds the next position.
// With at least n_layers micro-batches per chain every CTA always has one to work on.  Samples are
// independent (l.125), so chains never talk to each other.
//
// The GEMMs are "swap-AB" tcgen05.mma (cta_group::1, kind::f16, M = 128 output features, N = 16 samples,
// K = 16 per instruction): D[feature, sample] in TMEM columns 448..511, activations as the K-major
// SWIZZLE_128B B operand in shared memory, issued by one thread, completion by tcgen05.commit on an
// mbarrier, epilogues read TMEM with tcgen05.ld (lane = feature).  The KV rows of layer l for the chain's
// samples are written and read only by CTA l: the KV ring (fv_ring.cuh) holds nothing but KV rows and is
// refilled across micro-batch boundaries.
#include "fv_ring.cuh"
#include "fv_umma.cuh"

#include <cstdio>

namespace {
using namespace fvring;

constexpr int D = 128, DH = 16;
constexpr int NTHREADS = NWC * 32 + 32;       // compute warps + the KV producer warp
constexpr int MB_MAX = 16;                    // micro-batches per chain
constexpr int HS = D + 4;                     // fp32 residual row stride (words)
constexpr int QS2 = D + 4, KVS = 2 * D + 8;   // q fp32 / k|v bf16 row strides (fv_decode.cu)
constexpr int CH = fv_ring_ch(D);             // KV rows per ring chunk (host plan agrees)
constexpr int ROW_BYTES = 4 * D, CHUNK_BYTES = CH * ROW_BYTES;
constexpr int LPR = D / 8, LPH = DH / 8;
constexpr int TAB_C = 48, TAB_R = 48;
// tensor memory columns
constexpr uint32_t TC_WQKV = 0, TC_W1 = 192, TC_ACC = 448;

struct ChainArgs {
    int32_t B, R, MB, n_chains;
    const float* uniforms;
    int8_t* spins_out;
    float* logq;
    float* cond_p;
};

template <int RMAX>
struct ChainGeo {
    static constexpr int NSPLIT = NWC / RMAX > 1 ? NWC / RMAX : 1;     // warps per query row
    static constexpr int GR = NWC / NSPLIT;                            // rows attended at the same time
    static constexpr int SPS = D + 2 * LPR;                            // floats per split-partial slot
    static constexpr size_t off_w2 = 0;                                // [128 x 512] bf16, 8 K-blocks of 16 KB
    static constexpr size_t off_bact = 131072;                         // [16 x 128] bf16 B tile (LN output)
    static constexpr size_t off_u = off_bact + 4096;                   // union: FFN hidden B tile | q, k|v, split partials
    static constexpr size_t q_bytes = (size_t)RMAX * QS2 * 4, kv_bytes = (size_t)RMAX * KVS * 2;
    static constexpr size_t split_bytes = NSPLIT > 1 ? (size_t)RMAX * NSPLIT * SPS * 4 : 0;
    static constexpr size_t u_raw = q_bytes + kv_bytes + split_bytes > 16384 ? q_bytes + kv_bytes + split_bytes : 16384;
    static constexpr size_t u_bytes = (u_raw + 127) / 128 * 128;
    static constexpr size_t off_h = off_u + u_bytes;                   // two residual-stream buffers (the inbox)
    static constexpr size_t h_bytes = (size_t)RMAX * HS * 4;
    static constexpr size_t off_logq = off_h + 2 * h_bytes;            // double [MB_MAX][RMAX] (last CTA)
    static constexpr size_t off_tokin = off_logq + (size_t)MB_MAX * RMAX * 8;   // int [MB_MAX][RMAX] (CTA 0, written by the last CTA)
    static constexpr size_t off_misc = off_tokin + (size_t)MB_MAX * RMAX * 4;   // uniforms: float [2][RMAX]
    static constexpr size_t off_bar = off_misc + 2 * RMAX * 4;         // mbarriers and counters
    static constexpr int NSLOT_MAX = 10;
    static constexpr size_t bar_bytes = (2 * NSLOT_MAX + 2 + 2 + MB_MAX + 2) * 8 + 32;
    static constexpr size_t off_tab = (off_bar + bar_bytes + 15) / 16 * 16;
    static constexpr size_t tab_bytes = 2 * (TAB_C * 4 + TAB_R * 8);
    static constexpr size_t off_ring = (off_tab + tab_bytes + 127) / 128 * 128;
    static constexpr int NSLOT_RAW = (int)((SMEM_MAX - off_ring) / CHUNK_BYTES);
    static constexpr int NSLOT = NSLOT_RAW > NSLOT_MAX ? NSLOT_MAX : NSLOT_RAW;
    static constexpr size_t total = off_ring + (size_t)NSLOT * CHUNK_BYTES;
    static_assert(NSLOT >= 4, "KV ring too small");
    static_assert(off_u % 1024 == 0, "swizzled tiles need 1024-byte alignment");
};

// ---- cross-CTA waits carry a watchdog: a protocol error must end in a trap, never in a hung GPU ----------
__device__ __noinline__ void chain_timeout(int what) {
    printf("fv_chain_kernel: wait %d timed out (block %d thread %d)\n", what, (int)blockIdx.x, (int)threadIdx.x);
    __trap();
}
__device__ __forceinline__ void mbar_wait_cluster_wd(uint64_t* bar, uint32_t parity, int what) {
    const uint32_t addr = smem_u32(bar);
    uint32_t done;
    long long t0 = 0;
    int spins = 0;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}\n"
            : "=r"(done) : "r"(addr), "r"(parity) : "memory");
        if (!done && (++spins & 1023) == 0) {
            const long long now = clock64();
            if (t0 == 0) t0 = now;
            else if (now - t0 > 6000000000LL) chain_timeout(what);     // ~3 s
        }
    } while (!done);
}
__device__ __forceinline__ void st_peer_f32(uint32_t raddr, float v) {
    asm volatile("st.shared::cluster.f32 [%0], %1;\n" ::"r"(raddr), "f"(v) : "memory");
}
__device__ __forceinline__ void st_peer_s32(uint32_t raddr, int v) {
    asm volatile("st.shared::cluster.s32 [%0], %1;\n" ::"r"(raddr), "r"(v) : "memory");
}

template <int RMAX>
__global__ void __launch_bounds__(NTHREADS, 1)
fv_chain_kernel(const __grid_constant__ FvModelDev m, const __grid_constant__ ChainArgs a) {
    using G = ChainGeo<RMAX>;
    constexpr int NSPLIT = G::NSPLIT, GR = G::GR, SPS = G::SPS, NSLOT = G::NSLOT;
    constexpr int NC = RMAX;                                  // accumulator columns an epilogue reads (= samples)

    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char* sh_w2 = smem + G::off_w2;
    unsigned char* sh_bact = smem + G::off_bact;
    unsigned char* sh_bhid = smem + G::off_u;
    float* sh_q = reinterpret_cast<float*>(smem + G::off_u);
    __nv_bfloat16* sh_kv = reinterpret_cast<__nv_bfloat16*>(smem + G::off_u + G::q_bytes);
    float* sh_split = reinterpret_cast<float*>(smem + G::off_u + G::q_bytes + G::kv_bytes);
    float* sh_hbuf = reinterpret_cast<float*>(smem + G::off_h);
    double* sh_logq = reinterpret_cast<double*>(smem + G::off_logq);
    int* sh_tokin = reinterpret_cast<int*>(smem + G::off_tokin);
    float* sh_ubuf = reinterpret_cast<float*>(smem + G::off_misc);    // [2][RMAX] uniforms of the slot (last CTA)
    uint64_t* bar_full = reinterpret_cast<uint64_t*>(smem + G::off_bar);
    uint64_t* bar_empty = bar_full + G::NSLOT_MAX;
    uint64_t* bar_in = bar_empty + G::NSLOT_MAX;              // [2] residual rows of a micro-batch have arrived (from CTA l - 1)
    uint64_t* bar_free = bar_in + 2;                          // [2] CTA l + 1 has finished with its buffer
    uint64_t* bar_tok = bar_free + 2;                         // [MB_MAX] tokens of micro-batch mb have arrived (CTA 0)
    uint64_t* bar_mma = bar_tok + MB_MAX;                     // tcgen05.commit target
    uint64_t* bar_w = bar_mma + 1;                            // W_2 image has landed
    int* sh_app = reinterpret_cast<int*>(bar_w + 1);          // KV appends published so far (in slots)
    int* sh_issued = sh_app + 1;                              // ring chunks armed so far
    uint32_t* sh_tmem = reinterpret_cast<uint32_t*>(sh_app + 2);
    int32_t* tab_c = reinterpret_cast<int32_t*>(smem + G::off_tab);
    int2* tab_r = reinterpret_cast<int2*>(tab_c + 2 * TAB_C);
    unsigned char* ring = smem + G::off_ring;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int N = m.n_sites, NL = m.n_layers;
    const int l = (int)cluster_ctarank();                     // my layer
    const int chain = blockIdx.x / NL;
    const bool first = l == 0, last = l == NL - 1;
    const FvLayerDev& L = m.layer[l];
    // micro-batches of this chain: global micro-batch g = chain * MB + mb holds samples [g R, g R + R)
    const int g0 = chain * a.MB;
    int MBc = 0;                                              // the non-empty ones come first
    for (int mb = 0; mb < a.MB; ++mb) MBc += ((g0 + mb) * a.R < a.B);

    if (tid == 0) {
        for (int i = 0; i < NSLOT; ++i) { mbar_init(bar_full + i, 1); mbar_init(bar_empty + i, 1); }
        mbar_init(bar_in, 128); mbar_init(bar_in + 1, 128);
        mbar_init(bar_free, 1); mbar_init(bar_free + 1, 1);
        for (int i = 0; i < MB_MAX; ++i) mbar_init(bar_tok + i, 4);
        mbar_init(bar_mma, 4);
        mbar_init(bar_w, 1);
        *sh_app = 0;
        *sh_issued = 0;
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == 0) umma::tmem_alloc<512>(sh_tmem);
    umma::fence_before_sync();
    __syncthreads();
    umma::fence_after_sync();
    const uint32_t tm = *sh_tmem;
    cluster_sync_all();                                       // every CTA's barriers exist before anyone arrives on them

    // =============================== PRODUCER WARP ===============================
    // As in fv_decode.cu, but the ring carries only the KV rows of layer l for the micro-batches of the chain,
    // in slot order (t, mb): the rows of a slot are complete once slot (t - 1, mb) has appended, which this CTA
    // did MBc slots earlier, so the stream runs ahead across micro-batch boundaries.
    if (warp >= NWC) {
        if (lane == 0) {                                      // the layer's W_2 image: 8 K-blocks of [128 x 64] bf16
            constexpr int NKB = 8;
            mbar_arrive_expect_tx(bar_w, NKB * 16384u);
            const size_t per = ((size_t)FV_LP_HC * D + (size_t)D * FV_LP_HC) * 2;
            for (int j = 0; j < NKB; ++j)
                bulk_g2s(sh_w2 + j * 16384, L.img_ffn + j * per + (size_t)FV_LP_HC * D * 2, 16384u, bar_w);
        }
        uint64_t kv_pol = 0;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(kv_pol));
        constexpr int VW = NSLOT >= 16 ? 16 : (NSLOT >= 8 ? 8 : 4);
        uint32_t seq = 0;
        auto ready_prefix = [&](bool active, uint32_t slot, uint32_t par) {
            const bool ok = active && mbar_test_nb(bar_empty + slot, par ^ 1u);
            const unsigned int bm = __ballot_sync(0xffffffffu, ok);
            return bm == 0xffffffffu ? 32 : __ffs(~bm) - 1;
        };
        struct Plan { int nch, nn, nruns; const int32_t* cptr; const int2* rptr; };
        auto stage_plan = [&](int t) {
            Plan p;
            if (t >= N) { p.nch = p.nn = p.nruns = 0; p.cptr = nullptr; p.rptr = nullptr; return p; }
            const int cp0 = __ldg(m.chunk_ptr + t);
            p.nch = __ldg(m.chunk_ptr + t + 1) - cp0;
            p.nn = __ldg(m.mask_rowptr + t + 1) - 1 - __ldg(m.mask_rowptr + t);
            const int rp0 = __ldg(m.chunk_run_ptr + cp0);
            p.nruns = __ldg(m.chunk_run_ptr + cp0 + p.nch) - rp0;
            int32_t* tc = tab_c + (t & 1) * TAB_C;
            int2* tr = tab_r + (t & 1) * TAB_R;
            __syncwarp();
            if (p.nch + 1 <= TAB_C && p.nruns <= TAB_R) {
                for (int i = lane; i <= p.nch; i += 32) tc[i] = __ldg(m.chunk_run_ptr + cp0 + i) - rp0;
                for (int i = lane; i < p.nruns; i += 32) tr[i] = __ldg(m.runs + rp0 + i);
                __syncwarp();
                p.cptr = tc; p.rptr = tr;
            } else {
                p.cptr = m.chunk_run_ptr + cp0; p.rptr = m.runs;
            }
            return p;
        };
        Plan cur = stage_plan(0);
        for (int t = 0; t < N; ++t) {
            // the plan of step t + 1 may only replace the table of step t - 1 once every copy of step t - 1 has
            // been issued: it is staged after the loop over this step's micro-batches has started from `cur`
            const Plan nxt = stage_plan(t + 1);
            const int nch = cur.nch, nn = cur.nn;
            for (int mb = 0; mb < MBc; ++mb) {
                const int b_first = (g0 + mb) * a.R;
                const int n_own = min(a.R, a.B - b_first);
                const int total = n_own * nch;
                if (total > 0) {
                    const int need = (t - 1) * MBc + mb + 1;
                    while (ld_acquire_s32(sh_app) < need) __nanosleep(32);
                }
                const unsigned char* src_l = reinterpret_cast<const unsigned char*>(m.kv_s + ((size_t)b_first * NL + l) * m.kv_rows * (2 * D));
                for (int i0 = 0; i0 < total;) {
                    const int i = i0 + lane;
                    const uint32_t sq = seq + (uint32_t)i;
                    const uint32_t slot = sq % NSLOT, par = (sq / NSLOT) & 1u;
                    const int npre = ready_prefix(lane < VW && i < total, slot, par);
                    if (lane < npre) {
                        const int k = i / (GR * nch), rem = i - k * GR * nch;      // chunk-major inside a round of GR rows
                        const int nk = min(GR, n_own - k * GR);
                        const int c = rem / nk;
                        const int r = k * GR + (rem - c * nk);
                        const int rows = min(CH, nn - c * CH);
                        mbar_arrive_expect_tx(bar_full + slot, (uint32_t)rows * ROW_BYTES);
                        const unsigned char* src = src_l + (size_t)r * NL * m.kv_rows * ROW_BYTES;
                        unsigned char* dst = ring + (size_t)slot * CHUNK_BYTES;
                        const int j1 = cur.cptr[c + 1];
                        for (int j = cur.cptr[c]; j < j1; ++j) {
                            const int2 run = cur.rptr[j];
                            bulk_g2s_hint(dst + (size_t)(run.y >> 16) * ROW_BYTES, src + (size_t)run.x * ROW_BYTES,
                                          (uint32_t)(run.y & 0xffff) * ROW_BYTES, bar_full + slot, kv_pol);
                        }
                    }
                    __syncwarp();
                    i0 += npre;
                    if (lane == 0 && npre) st_release_s32(sh_issued, (int)(seq + (uint32_t)i0));
                }
                seq += (uint32_t)total;
            }
            cur = nxt;
        }
        cluster_sync_all();
        return;
    }

    // =============================== COMPUTE WARPS ===============================
    // ---- one-off: this layer's W_qkv and W_1 into tensor memory (lane = output feature, column = two K
    // elements), read back from the SWIZZLE_128B images fv_log_prob uses; W_2 arrives by TMA (producer) ----
    {
        const int q4 = warp & 3, row = q4 * 32 + lane;
        for (int tile = warp >> 2; tile < 7; tile += 4) {      // tiles 0-2: W_qkv rows 128 tile.., 3-6: W_1
            const unsigned char* img;
            int rr, rows_per_kb;
            if (tile < 3) { img = L.img_qkv; rr = tile * 128 + row; rows_per_kb = 3 * D; }
            else {
                const int hrow = (tile - 3) * 128 + row;         // hidden unit; image chunk j = hrow / 64
                const size_t per = ((size_t)FV_LP_HC * D + (size_t)D * FV_LP_HC) * 2;
                img = L.img_ffn + (size_t)(hrow / FV_LP_HC) * per; rr = hrow % FV_LP_HC; rows_per_kb = FV_LP_HC;
            }
            const uint32_t tbase = tm + ((uint32_t)(q4 * 32) << 16) + (tile < 3 ? TC_WQKV + tile * 64 : TC_W1 + (tile - 3) * 64);
#pragma unroll
            for (int kb = 0; kb < 2; ++kb)
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    const uint4 v = __ldg(reinterpret_cast<const uint4*>(img + (size_t)kb * rows_per_kb * 128 + umma::sw128_chunk(rr, c)));
                    umma::tmem_st4(tbase + kb * 32 + c * 4, v);
                }
        }
        asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory");
        umma::fence_before_sync();
        cbar();
        umma::fence_after_sync();
        mbar_wait(bar_w, 0);
    }

    const int rg = lane / LPR, sub = lane % LPR;
    const RingCtx rc{ring, bar_full, bar_empty, sh_issued};
    constexpr uint32_t idesc = umma::make_idesc_bf16(128, 16);
    const uint64_t bd_act = umma::make_desc_sw128(smem_u32(sh_bact));
    const uint64_t bd_hid = umma::make_desc_sw128(smem_u32(sh_bhid));
    const uint64_t ad_w2 = umma::make_desc_sw128(smem_u32(sh_w2));
    const uint32_t nxt_rank = (uint32_t)(l + 1), prv_rank = (uint32_t)(l - 1);
    uint32_t seq_base = 0, mma_par = 0;
    int ju = 0;                                               // slots done
    if (last) for (int i = tid; i < MB_MAX * RMAX; i += NWC * 32) sh_logq[i] = 0.0;

    for (int t = 0; t < N; ++t) {
        const int me0 = __ldg(m.mask_rowptr + t);
        const int nn = __ldg(m.mask_rowptr + t + 1) - 1 - me0;
        const int nch = (nn + CH - 1) / CH;
        for (int mb = 0; mb < MBc; ++mb, ++ju) {
            const int b_first = (g0 + mb) * a.R;
            const int n_own = min(a.R, a.B - b_first);
            const int buf = ju & 1;
            float* sh_h = sh_hbuf + buf * (RMAX * HS);
            // ---- input: residual rows from CTA l - 1, or (CTA 0) the embedding of the token the last CTA sent ----
            if (first) {
                if (t > 0) mbar_wait_cluster_wd(bar_tok + mb, (uint32_t)((t - 1) & 1), 1);
                for (int i = tid; i < RMAX * D; i += NWC * 32) {     // concatenated positional embedding (Eq. 15)
                    const int r = i / D, f = i - r * D;
                    const int dt = m.d_token;
                    const int tok = (t > 0 && r < n_own) ? sh_tokin[mb * RMAX + r] : 0;
                    sh_h[r * HS + f] = f < dt ? __ldg(m.tok_emb + tok * dt + f) : __ldg(m.posemb + (size_t)t * (D - dt) + (f - dt));
                }
                cbar();
            } else {
                mbar_wait_cluster_wd(bar_in + buf, (uint32_t)((ju >> 1) & 1), 2);
            }
            float* sh_u = sh_ubuf + buf * RMAX;
            if (last && tid < RMAX) sh_u[tid] = tid < n_own ? __ldg(a.uniforms + (size_t)(b_first + tid) * N + t) : 2.f;
            // ---- LN1 (Alg. 2 l.12) -> B tile ----------------------------------------------------------------------
            for (int r = warp; r < n_own; r += NWC) ln_row_btile<16>(sh_h + r * HS, L.ln1_g, L.ln1_b, m.ln_eps, false, sh_bact, r, lane);
            umma::fence_smem_to_async();
            cbar();
            // ---- q, k, v = W a + b (Eq. 2; Alg. 2 l.13): D[feature, sample] = W_qkv[tile] . a^T -------------------------
            // (four issuing threads, one per M-tile: a small tcgen05.mma costs its issuing thread ~45 cycles, the
            // tensor pipe ~10, so the tiles are issued concurrently from four warps)
            if (warp < 4 && lane == 0) {
                if (warp < 3) {
                    umma::fence_after_sync();
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks)
                        umma::mma_bf16_ts(tm + TC_ACC + warp * 16, tm + TC_WQKV + warp * 64 + ks * 8,
                                    bd_act + (uint64_t)(((ks >> 2) * 2048 + (ks & 3) * 32) >> 4), idesc, ks != 0);
                    umma::commit(bar_mma);
                } else {
                    mbar_arrive(bar_mma);
                }
            }
            mbar_wait(bar_mma, mma_par); mma_par ^= 1u;
            umma::fence_after_sync();
            if (warp < 12) {
                const int mt = warp >> 2, fl = (warp & 3) * 32 + lane;
                float v[NC];
                umma::tmem_ld_cols<NC>(tm + ((uint32_t)((warp & 3) * 32) << 16) + TC_ACC + mt * 16, v);
                const float bias = __ldg(L.bqkv + mt * D + fl);
                if (mt == 0) {
#pragma unroll
                    for (int s = 0; s < NC; ++s) sh_q[s * QS2 + fl] = v[s] + bias;
                } else {
#pragma unroll
                    for (int s = 0; s < NC; ++s) sh_kv[s * KVS + (mt - 1) * D + fl] = __float2bfloat16_rn(v[s] + bias);
                }
            }
            umma::fence_before_sync();
            cbar();
            // ---- append k_t, v_t to the KV pool as bf16 (Alg. 2 l.17; reading A2) ---------------------------------
            for (int i = tid; i < RMAX * (2 * D / 8); i += NWC * 32) {
                const int r = i / (2 * D / 8), ch = i - r * (2 * D / 8);
                if (r >= n_own) continue;
                const uint4 v = *reinterpret_cast<const uint4*>(sh_kv + r * KVS + ch * 8);
                __nv_bfloat16* dst = m.kv_s + (((size_t)(b_first + r) * NL + l) * m.kv_rows + t % m.kv_rows) * (2 * D) + ch * 8;
                *reinterpret_cast<uint4*>(dst) = v;
            }
            asm volatile("fence.proxy.async.global;\n" ::: "memory");   // the producer reads these rows by cp.async.bulk
            // ---- masked attention from the KV ring + residual (Eq. 3; Alg. 2 l.14-15) ---------------------------
            for (int task = warp; task < RMAX * NSPLIT; task += NWC) {
                const int r = task / NSPLIT, sp = task - r * NSPLIT;
                if (r >= n_own) continue;
                const float qs = kLog2e * rsqrtf((float)DH);
                const float* qrow = sh_q + r * QS2;
                const __nv_bfloat16* kvrow = sh_kv + r * KVS;
                float q[8], acc[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) q[j] = qrow[sub * 8 + j] * qs;
                float mm = -1e30f, ll = 0.f;
#pragma unroll
                for (int j = 0; j < 8; ++j) acc[j] = 0.f;
                if (sp == 0) {                       // row t itself, as the pool stores it (bf16)
                    float d = 0.f;
#pragma unroll
                    for (int j = 0; j < 8; ++j) d += q[j] * __bfloat162float(kvrow[sub * 8 + j]);
#pragma unroll
                    for (int o = 1; o < LPH; o <<= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
                    if (rg == 0) {
                        mm = d; ll = 1.f;
#pragma unroll
                        for (int j = 0; j < 8; ++j) acc[j] = __bfloat162float(kvrow[D + sub * 8 + j]);
                    }
                }
                for (int c = sp; c < nch; c += NSPLIT) {
                    const int kr = r / GR, nk = min(GR, n_own - kr * GR);
                    const uint32_t sq = seq_base + (uint32_t)(kr * GR * nch + c * nk + (r - kr * GR));
                    uint32_t slot;
                    const unsigned char* chunk = ring_acquire<NSLOT, CHUNK_BYTES>(rc, sq, slot);
                    attend_chunk<D, DH, CH>(chunk, min(CH, nn - c * CH), q, rg, sub, mm, ll, acc);
                    ring_release(rc, slot, lane);
                }
#pragma unroll
                for (int o = LPR; o < 32; o <<= 1) {       // merge the row groups of the warp
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
                if (lane < LPR) {
                    if (NSPLIT > 1) {
                        float* ps = sh_split + task * SPS;
                        ps[lane] = mm; ps[LPR + lane] = ll;
#pragma unroll
                        for (int j = 0; j < 8; ++j) ps[2 * LPR + lane * 8 + j] = acc[j];
                    } else {
                        const float inv = 1.0f / ll;
#pragma unroll
                        for (int j = 0; j < 8; ++j) sh_h[r * HS + lane * 8 + j] += acc[j] * inv;
                    }
                }
            }
            seq_base += (uint32_t)(n_own * nch);
            cbar();
            if (tid == 0) st_release_s32(sh_app, ju + 1);
            if (NSPLIT > 1) {                       // combine the split partials, fixed order
                for (int i = tid; i < RMAX * D; i += NWC * 32) {
                    const int r = i / D, f = i - r * D;
                    if (r >= n_own) continue;
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
                    sh_h[r * HS + f] += num / den;
                }
                cbar();
            }
            // ---- LN2 (Alg. 2 l.16; ln2_style 1 = Alg. 1 l.5) -> B tile ------------------------------------------
            for (int r = warp; r < n_own; r += NWC) ln_row_btile<16>(sh_h + r * HS, L.ln2_g, L.ln2_b, m.ln_eps, m.ln2_style == 1, sh_bact, r, lane);
            umma::fence_smem_to_async();
            cbar();
            // ---- FFN up-projection + exact GELU -> hidden B tile [16 x 512] ---------------------------------------
            if (warp < 4 && lane == 0) {
                umma::fence_after_sync();
#pragma unroll
                for (int ks = 0; ks < 8; ++ks)
                    umma::mma_bf16_ts(tm + TC_ACC + warp * 16, tm + TC_W1 + warp * 64 + ks * 8,
                                bd_act + (uint64_t)(((ks >> 2) * 2048 + (ks & 3) * 32) >> 4), idesc, ks != 0);
                umma::commit(bar_mma);
            }
            mbar_wait(bar_mma, mma_par); mma_par ^= 1u;
            umma::fence_after_sync();
            {
                const int mt = warp >> 2, jl = (warp & 3) * 32 + lane, j = mt * 128 + jl;     // hidden unit
                float v[NC];
                umma::tmem_ld_cols<NC>(tm + ((uint32_t)((warp & 3) * 32) << 16) + TC_ACC + mt * 16, v);
                const float b1 = __ldg(L.b1 + j);
                unsigned char* dst = sh_bhid + (j >> 6) * 2048 + (j & 7) * 2;
                const int c = (j & 63) >> 3;
#pragma unroll
                for (int s = 0; s < NC; ++s)
                    *reinterpret_cast<__nv_bfloat16*>(dst + umma::sw128_chunk(s, c)) = __float2bfloat16_rn(gelu_erf(v[s] + b1));
            }
            umma::fence_smem_to_async();
            umma::fence_before_sync();
            cbar();
            // ---- FFN down-projection (A = W_2 image in shared memory) + residual (Alg. 2 l.16) --------------------------
            // (K = 512 split over the four issuers: four partial accumulators, summed in the epilogue in fixed order)
            if (warp < 4 && lane == 0) {
                umma::fence_after_sync();
#pragma unroll
                for (int k8 = 0; k8 < 8; ++k8) {
                    const int ks = warp * 8 + k8;
                    umma::mma_bf16_ss_u(tm + TC_ACC + warp * 16, ad_w2 + (uint64_t)(((ks >> 2) * 16384 + (ks & 3) * 32) >> 4),
                                bd_hid + (uint64_t)(((ks >> 2) * 2048 + (ks & 3) * 32) >> 4), idesc, k8 != 0);
                }
                umma::commit(bar_mma);
            }
            mbar_wait(bar_mma, mma_par); mma_par ^= 1u;
            umma::fence_after_sync();
            if (warp < 4) {
                const int f = warp * 32 + lane;
                float v[NC];
                umma::tmem_ld_cols<NC>(tm + ((uint32_t)(warp * 32) << 16) + TC_ACC, v);
#pragma unroll
                for (int part = 1; part < 4; ++part) {
                    float v2[NC];
                    umma::tmem_ld_cols<NC>(tm + ((uint32_t)(warp * 32) << 16) + TC_ACC + part * 16, v2);
#pragma unroll
                    for (int s = 0; s < NC; ++s) v[s] += v2[s];
                }
                const float b2 = __ldg(L.b2 + f);
                if (!last) {
                    // the next CTA's buffer `buf` is free once it has finished slot ju - 2
                    if (ju >= 2) mbar_wait_cluster_wd(bar_free + buf, (uint32_t)(((ju >> 1) - 1) & 1), 3);
                    const uint32_t dst = map_to_peer(smem_u32(sh_h), nxt_rank);
#pragma unroll
                    for (int s = 0; s < NC; ++s)
                        if (s < n_own) st_peer_f32(dst + (uint32_t)(s * HS + f) * 4, sh_h[s * HS + f] + (v[s] + b2));
                    mbar_arrive_peer(map_to_peer(smem_u32(bar_in + buf), nxt_rank));      // release.cluster: after my stores
                } else {
#pragma unroll
                    for (int s = 0; s < NC; ++s)
                        if (s < n_own) sh_h[s * HS + f] += v[s] + b2;
                }
                umma::fence_before_sync();
                asm volatile("bar.sync 2, 128;\n" ::: "memory");     // the four epilogue warps
                if (last) {
                    // ---- output head: p(+1) = softmax(z)[1] = sigmoid(z1 - z0) (Alg. 2 l.20-22), draw, log q ---------
                    for (int r = warp; r < n_own; r += 4) {
                        const int b = b_first + r;
                        float d = 0.f;
#pragma unroll
                        for (int jj = 0; jj < D / 32; ++jj) d += sh_h[r * HS + lane * (D / 32) + jj] * __ldg(m.head_wd + lane * (D / 32) + jj);
                        d = warp_sum(d) + m.head_bd;
                        if (lane == 0) {
                            const float p = 1.0f / (1.0f + expf(-d));
                            const int up = sh_u[r] < p;                            // reading A10 (l.23)
                            a.spins_out[(size_t)b * N + t] = up ? 1 : -1;           // sigma = 2 s - 1 (l.25)
                            const float x = up ? -d : d;                           // log p(s) = -softplus(x)
                            const double lq = sh_logq[mb * RMAX + r] + (double)(-(fmaxf(x, 0.f) + log1pf(expf(-fabsf(x)))));
                            sh_logq[mb * RMAX + r] = lq;
                            if (t == N - 1) a.logq[b] = (float)lq;
                            if (a.cond_p) a.cond_p[(size_t)b * N + t] = p;
                            if (t + 1 < N) st_peer_s32(map_to_peer(smem_u32(sh_tokin + mb * RMAX + r), 0), up);
                        }
                    }
                    __syncwarp();
                    if (lane == 0 && t + 1 < N) mbar_arrive_peer(map_to_peer(smem_u32(bar_tok + mb), 0));
                    asm volatile("bar.sync 2, 128;\n" ::: "memory");  // all reads of this buffer are done
                }
                if (!first && tid == 0)                              // CTA l - 1 may refill this buffer
                    mbar_arrive_peer(map_to_peer(smem_u32(bar_free + buf), prv_rank));
            } else {
                umma::fence_before_sync();
            }
        }
    }
    cbar();
    umma::fence_before_sync();
    cluster_sync_all();                                       // no CTA leaves while a peer may still write to it
    if (warp == 0) {
        umma::fence_after_sync();
        umma::tmem_dealloc<512>(tm);
    }
}

}  // namespace

// ------------------------------------------------------------------------------ dispatch
template <int RMAX>
static cudaError_t launch_chain(const FvModelDev& m, const ChainArgs& a, cudaStream_t s) {
    auto kern = fv_chain_kernel<RMAX>;
    using G = ChainGeo<RMAX>;
    if (cudaError_t e = fv_smem_attr((const void*)kern, (int)G::total); e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)(a.n_chains * m.n_layers));
    cfg.blockDim = dim3(NTHREADS);
    cfg.dynamicSmemBytes = G::total;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)m.n_layers; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, m, a);
}

// Clusters of n_layers CTAs (one CTA per SM) the device can hold at once, per (device, n_layers).
static int chain_clusters(int n_layers) {
    static std::mutex mu;
    static std::map<std::pair<int, int>, int> cache;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    std::lock_guard<std::mutex> lock(mu);
    auto it = cache.find({dev, n_layers});
    if (it != cache.end()) return it->second;
    using G = ChainGeo<16>;
    int n = 0;
    if (fv_smem_attr((const void*)fv_chain_kernel<16>, (int)G::total) == cudaSuccess) {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)(n_layers * 64));
        cfg.blockDim = dim3(NTHREADS);
        cfg.dynamicSmemBytes = G::total;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = (unsigned)n_layers; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        if (cudaOccupancyMaxActiveClusters(&n, fv_chain_kernel<16>, &cfg) != cudaSuccess) { n = 0; (void)cudaGetLastError(); }
    }
    cache[{dev, n_layers}] = n;
    return n;
}

// fv_sample through the layer-pipelined clusters.  cudaErrorNotSupported when the shape is not covered
// (d = 128 with 16-wide heads, no W_O, at most 8 layers, batch small enough for 16 micro-batches of 16 per
// chain): the caller then uses the streaming kernel of fv_decode.cu.
static bool chain_geometry(const FvModelDev& m, int d_model, int d_head, int B, ChainArgs& a) {
    if (d_model != D || d_head != DH || m.has_wo || m.vocab > 2 || m.n_layers > 8 || !m.layer[0].img_ffn || !m.layer[0].img_qkv)
        return false;
    const int C = chain_clusters(m.n_layers);
    if (C <= 0) return false;
    const int NL = m.n_layers;
    int MB = (B + C * 16 - 1) / (C * 16);
    if (MB < NL) MB = NL;                            // a full pipeline: every CTA of the chain always has a micro-batch
    if (MB > MB_MAX) return false;
    int R = (B + C * MB - 1) / (C * MB);
    if (R < 1) R = 1;
    a.B = B; a.R = R; a.MB = MB;
    a.n_chains = (B + MB * R - 1) / (MB * R);
    return true;
}

bool fv_chain_supported(const FvModelDev& m, int d_model, int d_head, int B) {
    ChainArgs a{};
    return chain_geometry(m, d_model, d_head, B, a);
}

cudaError_t fv_launch_chain(const FvModelDev& m, int d_model, int d_head, const FvForwardArgs& fa, cudaStream_t s) {
    ChainArgs a{};
    if (!chain_geometry(m, d_model, d_head, fa.B, a)) return cudaErrorNotSupported;
    const int R = a.R;
    a.uniforms = fa.uniforms; a.spins_out = fa.spins_out; a.logq = fa.logq; a.cond_p = fa.cond_p;
    return R <= 8 ? launch_chain<8>(m, a, s) : launch_chain<16>(m, a, s);
}
