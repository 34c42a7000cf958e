// fv_internal.h -- shared declarations of the CUDA path (not part of the public ABI).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <map>
#include <mutex>
#include <string>
#include <utility>
#include <vector>

#define FV_MAX_LAYERS 16

// Hidden columns per chunk of the fused FFN of fv_logprob.cu (host image packer and kernel must agree).
constexpr int FV_LP_HC = 64;

// KV rows per ring chunk of the decode kernel (host plan and device kernel must agree).
#ifndef FV_DEC_CH128
#define FV_DEC_CH128 16
#endif
#define FV_DIRECT_MAX 6
constexpr int fv_ring_ch(int d_model) { return d_model >= 256 ? 8 : (d_model >= 128 ? FV_DEC_CH128 : 16); }

// Per-layer device pointers.  GEMM weights are bf16, pre-packed at fv_create_model time into
// mma.m16n8k16 A-fragment order: tile (mt, kt) of W[out,in] is 32 lanes x 16 B, contiguous,
// so one warp-wide 128-bit load fetches a whole 16x16 tile (see pack_mma_a in fv_api.cu).
struct FvLayerDev {
    const uint4* wqkv;  // [3d, d]  rows: Wq, Wk, Wv            (Eq. 2)
    const uint4* wo;    // [d, d] or nullptr                    (l.107: bypassed in the paper)
    const uint4* w1;    // [4d, d]
    const uint4* w2;    // [d, 4d]
    const float *bqkv, *bo, *b1, *b2;
    const float *ln1_g, *ln1_b, *ln2_g, *ln2_b;
    // fv_decode.cu keeps a layer's small fp32 parameters in shared memory; they are copied from this block of 13 d floats:
    // ln1_g | ln1_b | bqkv (3d) -- used up to the QKV epilogue -- then ln2_g | ln2_b | b1 (4d) | b2 | bo (zeros without W_O)
    const float* par;
    // fv_logprob.cu: pre-swizzled (SWIZZLE_128B, K-major) bf16 images, copied verbatim into shared memory
    const unsigned char* img_qkv;   // [3d rows x KP]
    const unsigned char* img_ffn;   // per 64-column hidden chunk j: W1_j [64 x KP] | W2_j [d x 64]
    const unsigned char* img_wo;    // [d rows x KP] (has_wo), same layout
    const unsigned char* img_w1t;   // fv_decode_tc.cu (d = 128): W1 per 128-row M-tile and 64-column K-block, [128 x 64] tiles of 16 KB
};

struct FvModelDev {
    int32_t n_sites, n_layers, has_wo, ln2_style;
    float ln_eps;
    int32_t d_token;
    const float* tok_emb;   // [2, d_token]
    const float* posemb;    // [N, d - d_token]
    const float* head_wd;   // [d]  = head_W[1] - head_W[0]   (softmax over 2 logits == sigmoid)
    float head_bd;          //      = head_b[1] - head_b[0]
    int32_t vocab;          // 2, or 16 / 256 with patch tokens: then the V-way head below is used instead
    const float* head_w;    // [vocab, d] fp32
    const float* head_b;    // [vocab]
    const int32_t* mask_rowptr;
    const int32_t* mask_col;
    // KV ring copy plan of fv_decode.cu (derived from the mask at fv_create_model): row t minus its own
    // entry is cut into chunks of fv_ring_ch(d) rows; each chunk is a list of runs of consecutive
    // positions, one cp.async.bulk per run.  run.x = first position, run.y = (row in chunk << 16) | length.
    const int32_t* chunk_ptr;      // [N+1]  chunks before step t
    const int32_t* chunk_run_ptr;  // [n_chunks+1]
    const int2* runs;
    // fv_decode.cu's own copy plan: the same, built without the step's first FV_DIRECT_MAX ISOLATED key positions (runs of
    // one row, e.g. the lattice neighbour two rows up) -- those rows the attention warps load straight from the pool, which
    // takes one small bulk copy per sample and layer-step off the TMA unit that paces the attention phase.
    const int32_t* d_chunk_ptr;    // [N+1]
    const int32_t* d_chunk_run_ptr;
    const int2* d_runs;
    const int32_t* d_nn;           // [N]  rows of step t that come through the ring
    const int32_t* d_dir;          // [N * FV_DIRECT_MAX]  physical rows loaded directly, -1 = none
    __nv_bfloat16* kv;      // [max_batch][n_layers][N][2d]  (K row then V row, bf16); fv_log_prob's pool
    // fv_sample's pool: the same array, or -- when every mask row is one run t-W..t (the band of Eq. S1) --
    // a ring-buffer window [max_batch][n_layers][kv_rows = W+1][2d] in which position p lives in row p % kv_rows
    // (the copy plan's run.x is then that physical row, runs cut at the wrap)
    __nv_bfloat16* kv_s;
    int32_t kv_rows;        // rows per (sample, layer) stream of kv_s: N, or W+1 in window mode
    // fv_logprob.cu block attention plan: per block of 32 queries the padded union of key positions and,
    // per 16-key step and query, a 16-bit allow mask
    const int32_t* att_blk_uptr;   // [att_nblk + 1] offsets into att_ukeys (multiples of 16)
    const int32_t* att_ukeys;
    const uint16_t* att_mask;      // [(total keys / 16) * 32]
    int32_t att_nblk;
    float* lp_h;            // fv_log_prob workspace: residual stream [max_batch * N, d] fp32 (or nullptr)
    float* lp_q;            //                        queries of the current layer, same shape
    FvLayerDev layer[FV_MAX_LAYERS];
};

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device setting: configure a kernel once per
// (kernel, device), under a lock (a process may hold models on several GPUs and call from several threads).
inline cudaError_t fv_smem_attr(const void* kern, int bytes) {
    static std::mutex mu;
    static std::map<std::pair<const void*, int>, int> done;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    int& have = done[std::make_pair(kern, dev)];
    if (have >= bytes) return cudaSuccess;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) have = bytes;
    return e;
}

// Optional per-kernel timing (fv_profile in flashvan.h): CUDA events around the launches of one kernel class,
// recorded on the launching stream; no-ops unless switched on.
enum { FV_K_SAMPLE = 0, FV_K_LP_QKV = 1, FV_K_LP_ATTN = 2, FV_K_LP_FFN = 3, FV_K_LP_HEAD = 4, FV_K_COUNT = 5 };
void fv_prof_begin(int kind, cudaStream_t s);
void fv_prof_end(int kind, cudaStream_t s);

enum { FV_MODE_SAMPLE = 0, FV_MODE_LOGPROB = 1 };

struct FvForwardArgs {
    int32_t mode;
    int32_t B;
    int32_t rows_per_group;      // SAMPLE: samples per group (<= 8*NT)
    int32_t n_groups;            // SAMPLE: number of sample groups
    int32_t samples_per_cta;     // LOGPROB: contiguous samples owned by one CTA
    const float* uniforms;       // SAMPLE
    const int8_t* spins_in;      // LOGPROB
    int8_t* spins_out;           // SAMPLE
    float* logq;
    float* cond_p;               // may be nullptr
};

// Launchers (fv_forward.cu / fv_energy.cu).  Return cudaError_t of the launch.
cudaError_t fv_launch_forward(const FvModelDev& m, int d_model, int d_head, int nt,
                              const FvForwardArgs& a, int grid, cudaStream_t s);
size_t fv_forward_smem_bytes(int d_model, int nt);
cudaError_t fv_launch_decode(const FvModelDev& m, int d_model, int d_head, int nt,
                             const FvForwardArgs& a, int n_sms, int cluster, cudaStream_t s);
cudaError_t fv_launch_decode_tc(const FvModelDev& m, int d_model, int d_head, int nt, const FvForwardArgs& a, int n_sms,
                                cudaStream_t s);
bool fv_chain_supported(const FvModelDev& m, int d_model, int d_head, int B);
cudaError_t fv_launch_chain(const FvModelDev& m, int d_model, int d_head, const FvForwardArgs& a, cudaStream_t s);
cudaError_t fv_launch_logprob_tc(const FvModelDev& m, int d_model, int d_head, int B, const int8_t* spins,
                                 float* logq, float* cond_p, int n_sms, int* n_launches, cudaStream_t s);
// fv_log_prob_static (flashvan.h): workspace of one call in a file-scope __device__ array of this size
constexpr size_t FV_LP_STATIC_BYTES = (size_t)64 << 20;
size_t fv_logprob_static_need(const FvModelDev& m, int d_model, int B);
cudaError_t fv_launch_logprob_tc_static(const FvModelDev& m, int d_model, int d_head, int B, const int8_t* spins,
                                        float* logq, float* cond_p, int n_sms, int* n_launches, cudaStream_t s);
void fv_pack_sw128(const float* W, int rows, int K, int ld, int KP, uint16_t* dst);
cudaError_t fv_launch_energy_csr(int B, int N, const int8_t* spins, const int32_t* rowptr,
                                 const int32_t* col, const float* val, int integer, float* E,
                                 cudaStream_t s);
cudaError_t fv_launch_energy_dense(int B, int N, const int8_t* spins, const float* J, float* E,
                                   cudaStream_t s);
cudaError_t fv_launch_free_energy(int B, const float* E, const float* logq, double T, double* out,
                                  cudaStream_t s);

cudaError_t fv_launch_tokens_to_spins(int B, int n_tokens, int P, const uint8_t* tokens, const int32_t* site_index,
                                      int8_t* spins, cudaStream_t s);
cudaError_t fv_launch_overlap(int B, int N, const int8_t* sa, const int8_t* sc, int32_t* dot, int32_t* hist,
                              cudaStream_t s);

cudaError_t fv_launch_lmc(int B, int N, int n_sweeps, int8_t* spins, const int32_t* rowptr, const int32_t* col,
                          const float* val, float beta, const float* ev, int32_t* accepted, cudaStream_t s);

// fv_mask.cu: rows[i] = ordered Markov boundary of vertex i, ascending; -1 and a
// message in err on a bad edge.
int fv_markov_rows(int32_t n, int64_t n_edges, const int32_t* edge_a, const int32_t* edge_b,
                   std::vector<std::vector<int32_t>>& rows, std::string& err);
