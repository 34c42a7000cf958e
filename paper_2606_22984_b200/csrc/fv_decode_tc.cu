// fv_decode_tc.cu -- the persistent KV-cached sampler of fv_sample (Alg. 2) for d = 128 with
// its projections on the 5th-generation tensor cores (tcgen05.mma, accumulators in tensor memory).
//
// Same organisation as fv_decode.cu: a CTA owns S <= 32 samples for all N steps and all layers (samples are
// independent, l.125), one PRODUCER warp streams one ordered sequence of 8 KB slots into a shared-memory ring
// (cp.async.bulk on mbarriers) -- the KV rows the mask names AND the layer's weights -- and 16 COMPUTE warps do
// LayerNorm, attention, epilogues, head and draw.  What differs is the GEMMs (Eq. 2 l.98-100; FFN l.346):
//   * "swap-AB": D[feature, sample] = W[tile] . act^T with M = 128 output features, N = 16 or 32 samples, K = 16 per
//     tcgen05.mma (cta_group::1, kind::f16, bf16 operands, fp32 accumulate in TMEM);
//   * the A operand is the weight stream itself: a weight TILE [128 features x 64 K] is a 16 KB SWIZZLE_128B image
//     copied by ONE bulk copy into two adjacent ring slots (half as many copies as the 8 KB fragment chunks of
//     fv_decode.cu) and read by the tensor core straight from the ring -- no warp ever loads a weight;
//   * four threads (lane 0 of compute warps 0-3) issue the MMAs of their accumulator tile as its weight tiles land
//     (a small tcgen05.mma costs its issuing thread ~45 cycles, the tensor pipe far less) and release the slots
//     with tcgen05.commit on the slots' "empty" barriers;
//   * activations are the K-major SWIZZLE_128B B tile the LayerNorm / GELU warps write; epilogues read TMEM with
//     tcgen05.ld (lane = feature) and add bias / apply GELU / add the residual.
// A tile needs two ADJACENT slots: when the running slot index would put it on the ring's last slot, a pad slot
// (armed and released without data) goes in front of it; both sides derive that from the running index alone.
#include "fv_ring.cuh"

namespace {
using namespace fvring;

constexpr int D = 128, DH = 16;
constexpr int NTHREADS = NWC * 32 + 32;       // compute warps + the producer warp
constexpr int HS = D + 4;                     // fp32 residual row stride (words)
constexpr int QS2 = D + 4, KVS = 2 * D + 8;   // q fp32 / k|v bf16 row strides
constexpr int CH = fv_ring_ch(D);             // KV rows per ring chunk (host plan agrees)
constexpr int ROW_BYTES = 4 * D, CHUNK_BYTES = CH * ROW_BYTES;
constexpr int LPR = D / 8, LPH = DH / 8;
constexpr int TAB_C = 48, TAB_R = 48;
constexpr int TILE_BYTES = 2 * CHUNK_BYTES;   // one weight tile [128 x 64] bf16
static_assert(CHUNK_BYTES == 8192, "a weight tile is two ring slots");
constexpr int NT_QKV = 6, NT_W1 = 8, NT_W2 = 8;   // weight tiles per matrix

template <int NT>
struct TcGeo {
    static constexpr int R = 8 * NT;                                   // samples (rows) per CTA
    static constexpr int NB = R <= 16 ? 16 : 32;                       // rows of a B tile = N of the MMAs
    static constexpr int NSPLIT = NWC / R > 1 ? NWC / R : 1;           // warps per query row
    static constexpr int GR = NWC / NSPLIT;                            // rows attended at the same time
    static constexpr int SPS = D + 2 * LPR;                            // floats per split-partial slot
    static constexpr size_t off_bact = 0;                              // [NB x 128] bf16 B tile (LN output)
    static constexpr size_t off_u = off_bact + (size_t)NB * 256;       // union: FFN hidden B tile [NB x 512] | q, k|v, split partials
    static constexpr size_t q_bytes = (size_t)R * QS2 * 4, kv_bytes = (size_t)R * KVS * 2;
    static constexpr size_t split_bytes = NSPLIT > 1 ? (size_t)R * NSPLIT * SPS * 4 : 0;
    static constexpr size_t u_raw = q_bytes + kv_bytes + split_bytes > (size_t)NB * 1024 ? q_bytes + kv_bytes + split_bytes : (size_t)NB * 1024;
    static constexpr size_t u_bytes = (u_raw + 127) / 128 * 128;
    static constexpr size_t off_h = off_u + u_bytes;                   // fp32 residual stream
    static constexpr size_t off_misc = off_h + (size_t)R * HS * 4;     // logq f64, logp, u, tok
    static constexpr size_t off_bar = (off_misc + (size_t)R * 20 + 15) / 16 * 16;
    static constexpr int NSLOT_MAX = 32;
    static constexpr size_t bar_bytes = (2 * NSLOT_MAX + 5) * 8 + 32;
    static constexpr size_t off_tab = (off_bar + bar_bytes + 15) / 16 * 16;
    static constexpr size_t tab_bytes = 2 * (TAB_C * 4 + TAB_R * 8);
    static constexpr size_t off_ring = (off_tab + tab_bytes + 1023) / 1024 * 1024;   // swizzled weight tiles: 1024-byte alignment
    static constexpr int NSLOT_RAW = (int)((SMEM_MAX - off_ring) / CHUNK_BYTES);
    static constexpr int NSLOT = (NSLOT_RAW > NSLOT_MAX ? NSLOT_MAX : NSLOT_RAW) & ~1;
    static constexpr size_t total = off_ring + (size_t)NSLOT * CHUNK_BYTES;
    static constexpr int TMEM_COLS = 4 * NB <= 64 ? 64 : 128;          // four accumulator tiles of NB columns
    static_assert(NSLOT >= 8, "ring too small");
    static_assert(off_u % 1024 == 0, "swizzled tiles need 1024-byte alignment");
};

// Position of the next weight tile in the slot sequence: skips the ring's last slot (a tile must not wrap).
template <int NSLOT>
__device__ __forceinline__ uint32_t tile_pos(uint32_t& seq, bool& padded) {
    padded = seq % NSLOT == NSLOT - 1;
    if (padded) ++seq;
    const uint32_t p = seq;
    seq += 2;
    return p;
}
template <int NSLOT>
__device__ __forceinline__ uint32_t skip_tiles(uint32_t seq, int n) {
    bool pd;
    for (int i = 0; i < n; ++i) (void)tile_pos<NSLOT>(seq, pd);
    return seq;
}

template <int NC>
__device__ __forceinline__ void ld_acc(uint32_t taddr, float (&v)[NC]) {
    if constexpr (NC == 32) umma::tmem_ld32(taddr, v);
    else umma::tmem_ld_cols<NC>(taddr, v);
}

template <int NT>
__global__ void __launch_bounds__(NTHREADS, 1)
fv_decode_tc_kernel(const __grid_constant__ FvModelDev m, const __grid_constant__ FvForwardArgs a) {
    using G = TcGeo<NT>;
    constexpr int R = G::R, NB = G::NB, NSPLIT = G::NSPLIT, GR = G::GR, SPS = G::SPS, NSLOT = G::NSLOT;
    constexpr int NC = R;                                     // accumulator columns an epilogue reads (= samples)

    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char* sh_bact = smem + G::off_bact;
    unsigned char* sh_bhid = smem + G::off_u;
    float* sh_q = reinterpret_cast<float*>(smem + G::off_u);
    __nv_bfloat16* sh_kv = reinterpret_cast<__nv_bfloat16*>(smem + G::off_u + G::q_bytes);
    float* sh_split = reinterpret_cast<float*>(smem + G::off_u + G::q_bytes + G::kv_bytes);
    float* sh_h = reinterpret_cast<float*>(smem + G::off_h);
    double* sh_logq = reinterpret_cast<double*>(smem + G::off_misc);
    float* sh_logp = reinterpret_cast<float*>(sh_logq + R);
    float* sh_u = sh_logp + R;
    int* sh_tok = reinterpret_cast<int*>(sh_u + R);
    uint64_t* bar_full = reinterpret_cast<uint64_t*>(smem + G::off_bar);
    uint64_t* bar_empty = bar_full + G::NSLOT_MAX;
    uint64_t* bar_mma = bar_empty + G::NSLOT_MAX;             // tcgen05.commit target of the GEMM phases
    int* sh_app = reinterpret_cast<int*>(bar_mma + 1);        // KV appends published so far
    int* sh_issued = sh_app + 1;                              // ring slots armed so far
    uint32_t* sh_tmem = reinterpret_cast<uint32_t*>(sh_app + 2);
    int32_t* tab_c = reinterpret_cast<int32_t*>(smem + G::off_tab);
    int2* tab_r = reinterpret_cast<int2*>(tab_c + 2 * TAB_C);
    unsigned char* ring = smem + G::off_ring;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int N = m.n_sites, NL = m.n_layers;

    if (tid == 0) {
        for (int i = 0; i < NSLOT; ++i) { mbar_init(bar_full + i, 1); mbar_init(bar_empty + i, 1); }
        mbar_init(bar_mma, 4);
        *sh_app = 0;
        *sh_issued = 0;
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == 0) umma::tmem_alloc<G::TMEM_COLS>(sh_tmem);
    umma::fence_before_sync();
    __syncthreads();
    umma::fence_after_sync();
    const uint32_t tm = *sh_tmem;
    const int n_walk = gridDim.x, walk0 = blockIdx.x;

    // =============================== PRODUCER WARP ===============================
    if (warp >= NWC) {
        uint64_t kv_pol = 0;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(kv_pol));
        constexpr int VW = NSLOT >= 32 ? 32 : (NSLOT >= 16 ? 16 : 8);
        uint32_t seq = 0;
        int it = 0;
        auto slot_free = [&](uint32_t sq) { return mbar_test_nb(bar_empty + sq % NSLOT, ((sq / NSLOT) & 1u) ^ 1u); };
        // n tiles of 16 KB, tile i at src + i * stride_b (+ the second-level offset for i odd): lane i takes tile i
        auto issue_tiles = [&](const unsigned char* src, int n, size_t stride_even, size_t stride_odd) {
            uint32_t s = seq, pos = 0;
            bool padded = false;
            for (int i = 0; i <= lane && i < n; ++i) pos = tile_pos<NSLOT>(s, padded);
            const uint32_t end = skip_tiles<NSLOT>(seq, n);
            for (int i0 = 0; i0 < n;) {
                const bool mine = lane >= i0 && lane < n;
                const bool ok = mine && slot_free(pos) && slot_free(pos + 1) && (!padded || slot_free(pos - 1));
                const unsigned int bm = __ballot_sync(0xffffffffu, ok || lane < i0 || lane >= n) >> i0;
                const int npre = min(n - i0, bm == (0xffffffffu >> i0) ? 32 - i0 : __ffs(~bm) - 1);
                if (mine && lane < i0 + npre) {
                    const uint32_t s0 = pos % NSLOT;
                    if (padded) mbar_arrive(bar_full + (pos - 1) % NSLOT);          // the pad slot: armed without data
                    mbar_arrive_expect_tx(bar_full + s0, (uint32_t)TILE_BYTES);
                    bulk_g2s(ring + (size_t)s0 * CHUNK_BYTES, src + (size_t)(lane >> 1) * stride_even + (size_t)(lane & 1) * stride_odd,
                             (uint32_t)TILE_BYTES, bar_full + s0);
                    mbar_arrive(bar_full + s0 + 1);                                 // second half: its bytes are counted on the first
                }
                __syncwarp();
                if (npre) {
                    i0 += npre;
                    const uint32_t upto = __shfl_sync(0xffffffffu, pos + 2, i0 - 1);
                    if (lane == 0) st_release_s32(sh_issued, (int)upto);
                }
            }
            seq = end;
        };
        for (int unit = walk0; unit < a.n_groups; unit += n_walk, ++it) {
            const int b_first = unit * a.rows_per_group;
            const int n_own = min(a.rows_per_group, a.B - b_first);
            struct Plan { int nch, nn, nruns; const int32_t* cptr; const int2* rptr; };
            auto stage_plan = [&](int t) {
                Plan p;
                if (t >= N) { p.nch = p.nn = p.nruns = 0; p.cptr = nullptr; p.rptr = nullptr; return p; }
                // the plan without the step's isolated rows (fv_internal.h: d_*): those the attention warps load themselves
                const int cp0 = __ldg(m.d_chunk_ptr + t);
                p.nch = __ldg(m.d_chunk_ptr + t + 1) - cp0;
                p.nn = __ldg(m.d_nn + t);
                const int rp0 = __ldg(m.d_chunk_run_ptr + cp0);
                p.nruns = __ldg(m.d_chunk_run_ptr + cp0 + p.nch) - rp0;
                int32_t* tc = tab_c + (t & 1) * TAB_C;
                int2* tr = tab_r + (t & 1) * TAB_R;
                __syncwarp();
                if (p.nch + 1 <= TAB_C && p.nruns <= TAB_R) {
                    for (int i = lane; i <= p.nch; i += 32) tc[i] = __ldg(m.d_chunk_run_ptr + cp0 + i) - rp0;
                    for (int i = lane; i < p.nruns; i += 32) tr[i] = __ldg(m.d_runs + rp0 + i);
                    __syncwarp();
                    p.cptr = tc; p.rptr = tr;
                } else {
                    p.cptr = m.d_chunk_run_ptr + cp0; p.rptr = m.d_runs;
                }
                return p;
            };
            Plan cur = stage_plan(0);
            for (int t = 0; t < N; ++t) {
                const Plan nxt = stage_plan(t + 1);
                const int nch = cur.nch, nn = cur.nn;
                const int total = n_own * nch;
                // chunk index -> (round, chunk, sample) without integer divisions in the per-lane path (they showed in the
                // kernel time of fv_decode.cu): q = umulhi(i, ceil(2^32 / d)) is exact for i, d < 2^16
                const uint32_t d_round = (uint32_t)(GR * (nch > 0 ? nch : 1)), inv_round = (uint32_t)((0x100000000ull + d_round - 1) / d_round);
                const uint32_t nk0 = (uint32_t)min(GR, n_own > 0 ? n_own : 1), inv_nk0 = (uint32_t)((0x100000000ull + nk0 - 1) / nk0);
                const uint32_t nk1 = (uint32_t)(n_own > GR ? n_own - GR : 1), inv_nk1 = (uint32_t)((0x100000000ull + nk1 - 1) / nk1);
                for (int l = 0; l < NL; ++l) {
                    const FvLayerDev& L = m.layer[l];
                    // W_qkv tile i = (M-tile i / 2, K-block i % 2) of the [3d x d] image: K-block slabs of 384 rows
                    issue_tiles(L.img_qkv, NT_QKV, (size_t)TILE_BYTES, (size_t)3 * D * 128);
                    if (total > 0) {
                        const int need = (it * N + (t - 1)) * NL + l + 1;       // rows < t of layer l are appended
                        while (ld_acquire_s32(sh_app) < need) __nanosleep(32);
                    }
                    const unsigned char* src_l = reinterpret_cast<const unsigned char*>(m.kv_s + ((size_t)b_first * NL + l) * m.kv_rows * (2 * D));
                    for (int i0 = 0; i0 < total;) {
                        const int i = i0 + lane;
                        const uint32_t sq = seq + (uint32_t)i;
                        const uint32_t slot = sq % NSLOT;
                        const bool ok = lane < VW && i < total && slot_free(sq);
                        const unsigned int bm = __ballot_sync(0xffffffffu, ok);
                        const int npre = bm == 0xffffffffu ? 32 : __ffs(~bm) - 1;
                        if (lane < npre) {
                            // chunk-major inside a round of GR samples
                            const bool small = total < 65536;
                            const int k = small ? (d_round == 1u ? i : (int)__umulhi((uint32_t)i, inv_round)) : i / (GR * nch);
                            const int rem = i - k * GR * nch;
                            const int nk = min(GR, n_own - k * GR);
                            const int c = !small ? rem / nk
                                                 : (k == 0 ? (nk0 == 1u ? rem : (int)__umulhi((uint32_t)rem, inv_nk0))
                                                           : (nk1 == 1u ? rem : (int)__umulhi((uint32_t)rem, inv_nk1)));
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
                    // W_1 tile i = (M-tile i / 2, K-block i % 2) of the M-tile-major image; W_2 tile j = K-block j
                    issue_tiles(L.img_w1t, NT_W1, (size_t)2 * TILE_BYTES, (size_t)TILE_BYTES);
                    issue_tiles(L.img_ffn + (size_t)FV_LP_HC * D * 2, NT_W2, (size_t)2 * 2 * TILE_BYTES, (size_t)2 * TILE_BYTES);
                }
                cur = nxt;
            }
        }
        return;
    }

    // =============================== COMPUTE WARPS ===============================
    const int rg = lane / LPR, sub = lane % LPR;
    const int q4 = warp & 3;                                  // TMEM lane quarter this warp may access
    const uint32_t tq = tm + ((uint32_t)(q4 * 32) << 16);
    const int fl = q4 * 32 + lane;                            // feature (TMEM lane) this thread reads in epilogues
    const RingCtx rc{ring, bar_full, bar_empty, sh_issued};
    constexpr uint32_t idesc = umma::make_idesc_bf16(128, NB);
    const uint64_t bd_act = umma::make_desc_sw128(smem_u32(sh_bact));
    const uint64_t bd_hid = umma::make_desc_sw128(smem_u32(sh_bhid));
    const uint64_t ad_ring = umma::make_desc_sw128(smem_u32(ring));
    uint32_t seq_base = 0, mma_par = 0;
    int it = 0;
    // One GEMM phase: the phase's n_tiles weight tiles sit at consecutive positions from seq_base; issuing thread w
    // (lane 0 of compute warp w < n_issuers) owns accumulator tile w and the weight tiles 2w, 2w + 1, which it feeds
    // to the tensor core as they land; all compute threads then wait for the four accumulator tiles.
    // (Measured: one barrier per accumulator tile, with each group of four warps running its epilogue and its share
    // of the next GEMM on its own, was slower -- cfg5 310 vs 292 ms, cfg4 85.8 vs 83.6 ms.)
    auto gemm_phase = [&](int n_tiles, int n_issuers, uint64_t b_base, bool k_split) {
        if (warp < 4 && lane == 0) {
            if (warp < n_issuers) {
                umma::fence_after_sync();
                uint32_t s = seq_base;
                bool first = true;
                for (int i = 0; i < n_tiles; ++i) {
                    bool padded;
                    const uint32_t p = tile_pos<NSLOT>(s, padded);
                    if ((i >> 1) != warp) continue;
                    while ((int)((uint32_t)ld_acquire_s32(sh_issued) - (p + 1)) <= 0) __nanosleep(20);
                    if (padded) mbar_arrive(bar_empty + (p - 1) % NSLOT);
                    const uint32_t slot = p % NSLOT;
                    mbar_wait(bar_full + slot, (p / NSLOT) & 1u);
                    umma::fence_after_sync();
                    // B operand: K-block i % 2 of the [NB x 128] activation tile, or (FFN 2) K-block i of the hidden tile
                    const uint64_t bd = b_base + (uint64_t)(((k_split ? i : (i & 1)) * (NB * 128)) >> 4);
                    const uint64_t ad = ad_ring + (uint64_t)((slot * CHUNK_BYTES) >> 4);
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks)
                        umma::mma_bf16_ss_u(tm + warp * NB, ad + (uint64_t)((ks * 32) >> 4), bd + (uint64_t)((ks * 32) >> 4), idesc,
                                            (first && ks == 0) ? 0u : 1u);
                    first = false;
                    umma::commit(bar_empty + slot);           // both slots of the tile are free once these MMAs have read it
                    umma::commit(bar_empty + slot + 1);
                }
                umma::commit(bar_mma);
            } else {
                mbar_arrive(bar_mma);
            }
        }
        seq_base = skip_tiles<NSLOT>(seq_base, n_tiles);
        mbar_wait(bar_mma, mma_par); mma_par ^= 1u;
        umma::fence_after_sync();
    };

    for (int unit = walk0; unit < a.n_groups; unit += n_walk, ++it) {
        const int b_first = unit * a.rows_per_group;
        const int n_own = min(a.rows_per_group, a.B - b_first);
        if (tid < R) { sh_tok[tid] = 0; sh_logq[tid] = 0.0; }
        for (int t = 0; t < N; ++t) {
            const int me0 = __ldg(m.mask_rowptr + t);
            const int nn = __ldg(m.d_nn + t);                        // rows that come through the ring
            int dir_pos[FV_DIRECT_MAX];                              // isolated key positions, loaded straight from the pool
#pragma unroll
            for (int i = 0; i < FV_DIRECT_MAX; ++i) dir_pos[i] = __ldg(m.d_dir + (size_t)t * FV_DIRECT_MAX + i);
            const int nch = (nn + CH - 1) / CH;
            if (tid < R) sh_u[tid] = tid < n_own ? __ldg(a.uniforms + (size_t)(b_first + tid) * N + t) : 2.f;
            cbar();
            // ---- concatenated positional embedding (Eq. 15, l.287-292) -------------------
            for (int i = tid; i < R * D; i += NWC * 32) {
                const int r = i / D, f = i - r * D;
                const int dt = m.d_token;
                sh_h[r * HS + f] = f < dt ? __ldg(m.tok_emb + sh_tok[r] * dt + f) : __ldg(m.posemb + (size_t)t * (D - dt) + (f - dt));
            }
            cbar();
            for (int l = 0; l < NL; ++l) {
                const FvLayerDev& L = m.layer[l];
                // ---- LN1 (Alg. 2 l.12) -> B tile -----------------------------------------------------------------
                for (int r = warp; r < n_own; r += NWC) ln_row_btile<NB>(sh_h + r * HS, L.ln1_g, L.ln1_b, m.ln_eps, false, sh_bact, r, lane);
                umma::fence_smem_to_async();
                cbar();
                // ---- q, k, v = W a + b (Eq. 2; Alg. 2 l.13): accumulator tile w = rows 128 w .. of [W_q; W_k; W_v] ----------
                gemm_phase(NT_QKV, 3, bd_act, false);
                if (warp < 12) {
                    const int mt = warp >> 2;
                    float v[NC];
                    ld_acc<NC>(tq + mt * NB, v);
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
                // ---- append k_t, v_t to the KV pool as bf16 (Alg. 2 l.17; reading A2) -------------------------------
                for (int i = tid; i < R * (2 * D / 8); i += NWC * 32) {
                    const int r = i / (2 * D / 8), ch = i - r * (2 * D / 8);
                    if (r >= n_own) continue;
                    const uint4 v = *reinterpret_cast<const uint4*>(sh_kv + r * KVS + ch * 8);
                    __nv_bfloat16* dst = m.kv_s + (((size_t)(b_first + r) * NL + l) * m.kv_rows + t % m.kv_rows) * (2 * D) + ch * 8;
                    *reinterpret_cast<uint4*>(dst) = v;
                }
                asm volatile("fence.proxy.async.global;\n" ::: "memory");   // the producer reads these rows by cp.async.bulk
                // ---- masked attention from the KV ring + residual (Eq. 3; Alg. 2 l.14-15) -------------------------
                for (int task = warp; task < R * NSPLIT; task += NWC) {
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
                    // isolated rows of the step, one per row group and load; the first set is requested before the ring's rows
                    constexpr int RPID = 32 / LPR;
                    auto dir_load = [&](int b0, uint4& k4, uint4& v4) {
                        int dpos = -1;
#pragma unroll
                        for (int i = 0; i < RPID; ++i) if (rg == i && b0 + i < FV_DIRECT_MAX) dpos = dir_pos[b0 + i < FV_DIRECT_MAX ? b0 + i : 0];
                        if (sp != 0) dpos = -1;
                        k4 = v4 = make_uint4(0u, 0u, 0u, 0u);
                        if (dpos >= 0) {
                            const __nv_bfloat16* dp = m.kv_s + (((size_t)(b_first + r) * NL + l) * m.kv_rows + dpos) * (2 * D) + sub * 8;
                            k4 = *reinterpret_cast<const uint4*>(dp);
                            v4 = *reinterpret_cast<const uint4*>(dp + D);
                        }
                        return dpos >= 0;
                    };
                    uint4 dk, dv;
                    const bool dok = dir_load(0, dk, dv);
                    for (int c = sp; c < nch; c += NSPLIT) {
                        const int kr = r / GR, nk = min(GR, n_own - kr * GR);
                        const uint32_t sq = seq_base + (uint32_t)(kr * GR * nch + c * nk + (r - kr * GR));
                        uint32_t slot;
                        const unsigned char* chunk = ring_acquire<NSLOT, CHUNK_BYTES>(rc, sq, slot);
                        attend_chunk<D, DH, CH>(chunk, min(CH, nn - c * CH), q, rg, sub, mm, ll, acc);
                        // release by data dependency instead of a proxy fence (fv_ring.cuh): every K word fed the scores behind
                        // ll, the V words fed acc[0..1] / [2..3] / [4..5] / [6..7]
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
                if (tid == 0) st_release_s32(sh_app, (it * N + t) * NL + l + 1);
                if (NSPLIT > 1) {                       // combine the split partials, fixed order
                    for (int i = tid; i < R * D; i += NWC * 32) {
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
                // ---- LN2 (Alg. 2 l.16; ln2_style 1 = Alg. 1 l.5) -> B tile ----------------------------------------
                for (int r = warp; r < n_own; r += NWC) ln_row_btile<NB>(sh_h + r * HS, L.ln2_g, L.ln2_b, m.ln_eps, m.ln2_style == 1, sh_bact, r, lane);
                umma::fence_smem_to_async();
                cbar();
                // ---- FFN up-projection + exact GELU -> hidden B tile [NB x 512] ------------------------------------
                gemm_phase(NT_W1, 4, bd_act, false);
                {
                    const int mt = warp >> 2, j = mt * 128 + fl;                         // hidden unit = K index of the down-projection
                    float v[NC];
                    ld_acc<NC>(tq + mt * NB, v);
                    const float b1 = __ldg(L.b1 + j);
                    unsigned char* dst = sh_bhid + (j >> 6) * (NB * 128) + (j & 7) * 2;
                    const int c = (j & 63) >> 3;
#pragma unroll
                    for (int s = 0; s < NC; s += 2) {
                        const uint32_t g2 = gelu_erfc_x2(v[s] + b1, v[s + 1] + b1);      // samples s, s + 1 -> rows s, s + 1
                        *reinterpret_cast<uint16_t*>(dst + umma::sw128_chunk(s, c)) = (uint16_t)(g2 & 0xffffu);
                        *reinterpret_cast<uint16_t*>(dst + umma::sw128_chunk(s + 1, c)) = (uint16_t)(g2 >> 16);
                    }
                }
                umma::fence_smem_to_async();
                umma::fence_before_sync();
                cbar();
                // ---- FFN down-projection: K = 512 split over the four issuers (tiles 2w, 2w + 1 = K-blocks) + residual ----
                gemm_phase(NT_W2, 4, bd_hid, true);
                if (warp < 4) {
                    float v[NC];
                    ld_acc<NC>(tq, v);
#pragma unroll
                    for (int part = 1; part < 4; ++part) {
                        float v2[NC];
                        ld_acc<NC>(tq + part * NB, v2);
#pragma unroll
                        for (int s = 0; s < NC; ++s) v[s] += v2[s];
                    }
                    const float b2 = __ldg(L.b2 + fl);
#pragma unroll
                    for (int s = 0; s < NC; ++s)
                        if (s < n_own) sh_h[s * HS + fl] += v[s] + b2;
                }
                umma::fence_before_sync();
                cbar();
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
    umma::fence_before_sync();
    cbar();
    if (warp == 0) {
        umma::fence_after_sync();
        umma::tmem_dealloc<G::TMEM_COLS>(tm);
    }
}

}  // namespace

// ------------------------------------------------------------------------------ dispatch
template <int NT>
static cudaError_t launch_tc(const FvModelDev& m, const FvForwardArgs& a, int n_sms, cudaStream_t s) {
    auto kern = fv_decode_tc_kernel<NT>;
    using G = TcGeo<NT>;
    if (cudaError_t e = fv_smem_attr((const void*)kern, (int)G::total); e != cudaSuccess) return e;
    kern<<<a.n_groups < n_sms ? a.n_groups : n_sms, NTHREADS, G::total, s>>>(m, a);
    return cudaGetLastError();
}

// fv_sample with the projections on tcgen05: d = 128, 16-wide heads, no W_O (cudaErrorNotSupported otherwise: the
// caller falls back to fv_decode.cu).  nt = n8-tiles of samples per CTA as for fv_launch_decode.
cudaError_t fv_launch_decode_tc(const FvModelDev& m, int d_model, int d_head, int nt, const FvForwardArgs& a, int n_sms,
                                cudaStream_t s) {
    if (d_model != D || d_head != DH || m.has_wo || !m.layer[0].img_qkv || !m.layer[0].img_w1t) return cudaErrorNotSupported;
    switch (nt) {
        case 1: return launch_tc<1>(m, a, n_sms, s);
        case 2: return launch_tc<2>(m, a, n_sms, s);
        case 4: return launch_tc<4>(m, a, n_sms, s);
        default: return cudaErrorNotSupported;
    }
}
