// fv_energy.cu -- batched Ising energies and the F_q reduction for sm_100a.
//   EA lattices: E_b = -sum_bonds J_ij s_i s_j, CSR gather-reduce      (Eq. 8)
//   dense SK   : E_b = -sum_{i<j} J_ij s_i s_j                          (Eq. 6)
//   F_q        : mean_b(E_b + T log q_b) and its std                    (Eq. 5)
// All reductions use a fixed tree (shuffle, then shared memory) => bit-reproducible.
#include "fv_internal.h"
#include "fv_umma.cuh"

namespace {

template <typename T>
__device__ __forceinline__ T warp_reduce(T v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <typename T, int NW>
__device__ __forceinline__ T block_reduce(T v, T* scratch) {
    v = warp_reduce(v);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) scratch[warp] = v;
    __syncthreads();
    T r = (threadIdx.x < NW) ? scratch[threadIdx.x] : T(0);
    if (warp == 0) r = warp_reduce(r);
    if (threadIdx.x == 0) scratch[0] = r;
    __syncthreads();
    return scratch[0];
}

// One CTA per sample.  The sample's N spins are staged in shared memory (coalesced 1-byte
// loads), then thread i walks the bonds of sites i, i+256, ...; the couplings (a few KB to
// a few hundred KB) stay L1/L2 resident across CTAs.  +-J: int32 accumulation, exact.
template <bool INTEGER>
__global__ void __launch_bounds__(256) energy_csr_kernel(int N, const int8_t* __restrict__ spins,
                                                         const int32_t* __restrict__ rowptr,
                                                         const int32_t* __restrict__ col,
                                                         const float* __restrict__ val, float* __restrict__ E) {
    extern __shared__ int8_t sh_s[];
    __shared__ float red_f[8];
    __shared__ int red_i[8];
    const int b = blockIdx.x;
    const int8_t* s = spins + (size_t)b * N;
    for (int i = threadIdx.x; i < N; i += 256) sh_s[i] = s[i];
    __syncthreads();
    float accf = 0.f;
    int acci = 0;
    for (int i = threadIdx.x; i < N; i += 256) {
        const int si = sh_s[i];
        const int e0 = __ldg(rowptr + i), e1 = __ldg(rowptr + i + 1);
        for (int e = e0; e < e1; ++e) {
            const int sj = sh_s[__ldg(col + e)];
            if (INTEGER) acci += (int)__ldg(val + e) * si * sj;
            else accf += __ldg(val + e) * (float)(si * sj);
        }
    }
    if (INTEGER) {
        const int t = block_reduce<int, 8>(acci, red_i);
        if (threadIdx.x == 0) E[b] = -(float)t;
    } else {
        const float t = block_reduce<float, 8>(accf, red_f);
        if (threadIdx.x == 0) E[b] = -t;
    }
}

// Dense SK, CUDA-core revision: one warp per sample walks the strict upper triangle of J
// (fp32, L2 resident), lanes stride over j.  Superseded by the tensor-core s^T J s path for
// large batches.
__global__ void __launch_bounds__(256) energy_dense_kernel(int B, int N, const int8_t* __restrict__ spins,
                                                           const float* __restrict__ J, float* __restrict__ E) {
    extern __shared__ int8_t sh_s[];                    // [8][N]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int b = blockIdx.x * 8 + warp;
    if (b >= B) return;
    int8_t* s = sh_s + (size_t)warp * N;
    for (int i = lane; i < N; i += 32) s[i] = spins[(size_t)b * N + i];
    __syncwarp();
    float acc = 0.f;
    for (int i = 0; i < N - 1; ++i) {
        const float* row = J + (size_t)i * N;
        float part = 0.f;
        for (int j = i + 1 + lane; j < N; j += 32) part += __ldg(row + j) * (float)s[j];
        acc += part * (float)s[i];
    }
    acc = warp_reduce(acc);
    if (lane == 0) E[b] = -acc;
}

// Dense SK on the tensor cores (Eq. 6): T = S J as a bf16 tcgen05 GEMM with fp32
// accumulation in tensor memory, then E_b = -1/2 sum_j T[b,j] s_bj in the epilogue.
//   A = S  [128 samples x K = sites i], spins +-1 are exact in bf16, K-major, SWIZZLE_128B;
//   B = J  [128 sites j  x K = sites i] (J is symmetric, so row j of J is column j), split on the
//       fly into three bf16 terms hi + mid + lo (~24 mantissa bits: the 1e-4 relative bar needs
//       more than bf16's 8) that accumulate into the same TMEM columns.
// One CTA per 128 samples; j-tiles of 128 columns; per 64-wide K-block the four warps stage the
// operand tiles in shared memory, one thread issues 4 (K = 16) MMAs per term, tcgen05.commit on
// an mbarrier releases the tiles.  The whole GEMM is ~13 GFLOP on cfg3 (launch-latency sized), so
// the kernel favours simplicity over overlap.
__global__ void __launch_bounds__(128, 1) energy_dense_umma_kernel(int B, int N, const int8_t* __restrict__ spins,
                                                                   const float* __restrict__ J, float* __restrict__ E) {
    extern __shared__ __align__(1024) unsigned char esm_raw[];
    unsigned char* esm = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(esm_raw) + 1023) & ~(uintptr_t)1023);
    unsigned char* sA = esm;                    // [128 x 64] bf16, 16 KB
    unsigned char* sB = esm + 16384;            // 3 terms x [128 x 64] bf16, 48 KB
    __shared__ uint64_t bar;
    __shared__ uint32_t tmem_slot;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int b0 = blockIdx.x * 128;
    if (tid == 0) { umma::mbar_init(&bar, 1); umma::fence_mbar_init(); }
    if (warp == 0) umma::tmem_alloc<128>(&tmem_slot);
    umma::fence_before_sync();
    __syncthreads();
    umma::fence_after_sync();
    const uint32_t tmem = tmem_slot;
    const uint32_t idesc = umma::make_idesc_bf16(128, 128);
    const int KB = (N + 63) / 64, JT = (N + 127) / 128;
    uint32_t phase = 0;
    float e_acc = 0.f;
    const int my_b = b0 + tid;                  // epilogue: thread <-> TMEM lane <-> sample
    for (int jt = 0; jt < JT; ++jt) {
        for (int kb = 0; kb < KB; ++kb) {
            // ---- stage A: 128 samples x 64 sites; thread (r = tid) converts its row ------------
            {
                const int b = b0 + tid;
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    uint32_t w[4];
#pragma unroll
                    for (int h = 0; h < 4; ++h) {
                        const int i = kb * 64 + c * 8 + 2 * h;
                        const float x0 = (b < B && i < N) ? (float)spins[(size_t)b * N + i] : 0.f;
                        const float x1 = (b < B && i + 1 < N) ? (float)spins[(size_t)b * N + i + 1] : 0.f;
                        __nv_bfloat162 v = __floats2bfloat162_rn(x0, x1);
                        w[h] = *reinterpret_cast<uint32_t*>(&v);
                    }
                    *reinterpret_cast<uint4*>(sA + umma::sw128_chunk(tid, c)) = make_uint4(w[0], w[1], w[2], w[3]);
                }
            }
            // ---- stage B: rows j of J, 64 columns i, three bf16 split terms ----------------------
            for (int idx = tid; idx < 128 * 8; idx += 128) {
                const int r = idx >> 3, c = idx & 7;       // consecutive threads: consecutive 32 B of a row
                const int j = jt * 128 + r;
                uint32_t hi[4], mid[4], lo[4];
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    float x[2];
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        const int i = kb * 64 + c * 8 + 2 * h + q;
                        x[q] = (j < N && i < N) ? __ldg(J + (size_t)j * N + i) : 0.f;
                    }
                    const __nv_bfloat16 h0 = __float2bfloat16_rn(x[0]), h1 = __float2bfloat16_rn(x[1]);
                    const float r0 = x[0] - __bfloat162float(h0), r1 = x[1] - __bfloat162float(h1);
                    const __nv_bfloat16 m0 = __float2bfloat16_rn(r0), m1 = __float2bfloat16_rn(r1);
                    const __nv_bfloat16 l0 = __float2bfloat16_rn(r0 - __bfloat162float(m0));
                    const __nv_bfloat16 l1 = __float2bfloat16_rn(r1 - __bfloat162float(m1));
                    __nv_bfloat162 vh(h0, h1), vm(m0, m1), vl(l0, l1);
                    hi[h] = *reinterpret_cast<uint32_t*>(&vh);
                    mid[h] = *reinterpret_cast<uint32_t*>(&vm);
                    lo[h] = *reinterpret_cast<uint32_t*>(&vl);
                }
                const uint32_t off = umma::sw128_chunk(r, c);
                *reinterpret_cast<uint4*>(sB + off) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
                *reinterpret_cast<uint4*>(sB + 16384 + off) = make_uint4(mid[0], mid[1], mid[2], mid[3]);
                *reinterpret_cast<uint4*>(sB + 32768 + off) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
            }
            umma::fence_smem_to_async();
            __syncthreads();
            if (tid == 0) {
                umma::fence_after_sync();
                const uint32_t a0 = umma::smem_u32(sA), bb = umma::smem_u32(sB);
#pragma unroll
                for (int term = 0; term < 3; ++term) {
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks) {
                        umma::mma_bf16_ss(tmem, umma::make_desc_sw128(a0 + ks * 32),
                                          umma::make_desc_sw128(bb + term * 16384 + ks * 32), idesc,
                                          (kb | term | ks) != 0);
                    }
                }
                umma::commit(&bar);
            }
            umma::mbar_wait(&bar, phase);          // MMAs done: tiles may be overwritten, TMEM readable
            phase ^= 1;
        }
        // ---- epilogue of this j-tile: E_b += sum_j T[b,j] s_bj ------------------------------------
        umma::fence_after_sync();
#pragma unroll 1
        for (int cb = 0; cb < 4; ++cb) {
            float v[32];
            umma::tmem_ld32(tmem + ((uint32_t)(warp * 32) << 16) + cb * 32, v);
            if (my_b < B) {
#pragma unroll
                for (int q = 0; q < 32; ++q) {
                    const int j = jt * 128 + cb * 32 + q;
                    if (j < N) e_acc += v[q] * (float)spins[(size_t)my_b * N + j];
                }
            }
        }
        umma::fence_before_sync();
        __syncthreads();                            // all TMEM reads done before the next tile's MMAs
    }
    if (my_b < B) E[my_b] = -0.5f * e_acc;
    __syncthreads();
    if (warp == 0) umma::tmem_dealloc<128>(tmem);
}

__global__ void __launch_bounds__(1024) free_energy_kernel(int B, const float* __restrict__ E,
                                                           const float* __restrict__ logq, double T,
                                                           double* __restrict__ out) {
    __shared__ double red[32];
    double s = 0.0;
    for (int i = threadIdx.x; i < B; i += 1024) s += (double)E[i] + T * (double)logq[i];
    const double mean = block_reduce<double, 32>(s, red) / B;
    double v = 0.0;
    for (int i = threadIdx.x; i < B; i += 1024) {
        const double d = (double)E[i] + T * (double)logq[i] - mean;
        v += d * d;
    }
    const double var = block_reduce<double, 32>(v, red) / B;
    // out[2], out[3]: what a multi-rank merge needs (count and sum of squared deviations, shard.py)
    if (threadIdx.x == 0) { out[0] = mean; out[1] = sqrt(var); out[2] = (double)B; out[3] = var * B; }
}

}  // namespace

cudaError_t fv_launch_energy_csr(int B, int N, const int8_t* spins, const int32_t* rowptr, const int32_t* col,
                                 const float* val, int integer, float* E, cudaStream_t s) {
    const size_t smem = (size_t)N;
    if (smem > 200 * 1024) return cudaErrorInvalidValue;
    if (integer) {
        if (smem > 48 * 1024) cudaFuncSetAttribute(energy_csr_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        energy_csr_kernel<true><<<B, 256, smem, s>>>(N, spins, rowptr, col, val, E);
    } else {
        if (smem > 48 * 1024) cudaFuncSetAttribute(energy_csr_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        energy_csr_kernel<false><<<B, 256, smem, s>>>(N, spins, rowptr, col, val, E);
    }
    return cudaGetLastError();
}

cudaError_t fv_launch_energy_dense(int B, int N, const int8_t* spins, const float* J, float* E, cudaStream_t s) {
    if (N >= 32) {                                  // tensor-core s^T J s (tcgen05, 3-term bf16 split of J)
        const int smem_tc = 65536 + 1024;
        if (cudaError_t e = fv_smem_attr((const void*)energy_dense_umma_kernel, smem_tc); e != cudaSuccess) return e;
        energy_dense_umma_kernel<<<(B + 127) / 128, 128, smem_tc, s>>>(B, N, spins, J, E);
        return cudaGetLastError();
    }
    const size_t smem = (size_t)8 * N;
    if (smem > 200 * 1024) return cudaErrorInvalidValue;
    if (smem > 48 * 1024) cudaFuncSetAttribute(energy_dense_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    energy_dense_kernel<<<(B + 7) / 8, 256, smem, s>>>(B, N, spins, J, E);
    return cudaGetLastError();
}

// Replica overlap (Eq. 9): dot[b] = sum_i a[b,i] * c[b,i], exact in int32; one warp per sample,
// 16 spins per lane and load, products and partial sums by dp4a; hist[(dot + N) / 2] += 1 (integer atomics:
// the result does not depend on their order).
__global__ void __launch_bounds__(256) overlap_kernel(int B, int N, const int8_t* __restrict__ sa, const int8_t* __restrict__ sc,
                                                      int32_t* __restrict__ dot, int32_t* __restrict__ hist) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= B) return;
    const int8_t* a = sa + (size_t)warp * N;
    const int8_t* c = sc + (size_t)warp * N;
    int acc = 0;
    // rows start at arbitrary byte offsets when N is not a multiple of 16: vector loads only if both are aligned
    const bool vec = ((reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(c)) & 15) == 0;
    const int nv = vec ? N / 16 : 0;
    for (int i = lane; i < nv; i += 32) {
        const int4 x = __ldg(reinterpret_cast<const int4*>(a) + i), y = __ldg(reinterpret_cast<const int4*>(c) + i);
        acc = __dp4a(x.x, y.x, acc); acc = __dp4a(x.y, y.y, acc);
        acc = __dp4a(x.z, y.z, acc); acc = __dp4a(x.w, y.w, acc);
    }
    for (int i = nv * 16 + lane; i < N; i += 32) acc += (int)a[i] * (int)c[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) {
        dot[warp] = acc;
        if (hist) atomicAdd(hist + ((acc + N) >> 1), 1);
    }
}

cudaError_t fv_launch_overlap(int B, int N, const int8_t* sa, const int8_t* sc, int32_t* dot, int32_t* hist, cudaStream_t s) {
    if (hist) {
        cudaError_t e = cudaMemsetAsync(hist, 0, sizeof(int32_t) * (size_t)(N + 1), s);
        if (e != cudaSuccess) return e;
    }
    overlap_kernel<<<(B + 7) / 8, 256, 0, s>>>(B, N, sa, sc, dot, hist);
    return cudaGetLastError();
}

// Local Monte Carlo refinement (Metropolis single-spin flips in site order, the
// acceptance test beta * dE < e with a caller-supplied exponential variate e -- no transcendental, so every
// decision is one fp32 multiplication and one comparison).  A sweep is sequential in the sites, so one warp owns
// one sample: its spins live in shared memory for all sweeps, lane 0 walks the sites (h_i accumulated in fp32 in
// adjacency order), the warp loads and stores the row with coalesced 16-byte accesses.
__global__ void __launch_bounds__(256) lmc_kernel(int B, int N, int n_sweeps, int8_t* __restrict__ spins,
                                                  const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                                                  const float* __restrict__ val, float beta, const float* __restrict__ ev,
                                                  int32_t* __restrict__ accepted, int row_stride) {
    extern __shared__ __align__(16) int8_t lmc_rows[];
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int b = blockIdx.x * (blockDim.x >> 5) + wib;
    if (b >= B) return;
    int8_t* s = lmc_rows + (size_t)wib * row_stride;
    int8_t* g = spins + (size_t)b * N;
    for (int i = lane; i < N; i += 32) s[i] = g[i];
    __syncwarp();
    int acc = 0;
    if (lane == 0) {
        const float* e = ev + (size_t)b * n_sweeps * N;
        for (int k = 0; k < n_sweeps; ++k, e += N) {
            int p0 = __ldg(rowptr);
            for (int i = 0; i < N; ++i) {
                const int p1 = __ldg(rowptr + i + 1);
                float h = 0.f;
                for (int p = p0; p < p1; ++p) h = __fadd_rn(h, __fmul_rn(__ldg(val + p), (float)s[__ldg(col + p)]));
                p0 = p1;
                const float dE = __fmul_rn(__fmul_rn(2.0f, (float)s[i]), h);
                if (__fmul_rn(beta, dE) < __ldg(e + i)) {
                    s[i] = -s[i];
                    ++acc;
                }
            }
        }
        if (accepted) accepted[b] = acc;
    }
    __syncwarp();
    for (int i = lane; i < N; i += 32) g[i] = s[i];
}

cudaError_t fv_launch_lmc(int B, int N, int n_sweeps, int8_t* spins, const int32_t* rowptr, const int32_t* col,
                          const float* val, float beta, const float* ev, int32_t* accepted, cudaStream_t s) {
    const int row_stride = (N + 15) / 16 * 16;
    int warps = 8;
    while (warps > 1 && (size_t)warps * row_stride > 48 * 1024) warps >>= 1;
    if ((size_t)warps * row_stride > 48 * 1024) return cudaErrorInvalidValue;
    lmc_kernel<<<(B + warps - 1) / warps, warps * 32, (size_t)warps * row_stride, s>>>(B, N, n_sweeps, spins, rowptr, col, val,
                                                                                      beta, ev, accepted, row_stride);
    return cudaGetLastError();
}

// Patch tokens -> lattice spins: one thread per (sample, token), P byte stores.
__global__ void tokens_to_spins_kernel(int B, int n_tokens, int P, const uint8_t* __restrict__ tokens,
                                       const int32_t* __restrict__ site_index, int8_t* __restrict__ spins) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)B * n_tokens) return;
    const int n = (int)(i % n_tokens);
    const long long b = i / n_tokens;
    const unsigned tok = tokens[i];
    for (int k = 0; k < P; ++k) spins[b * n_tokens * P + __ldg(site_index + n * P + k)] = ((tok >> k) & 1u) ? 1 : -1;
}

cudaError_t fv_launch_tokens_to_spins(int B, int n_tokens, int P, const uint8_t* tokens, const int32_t* site_index,
                                      int8_t* spins, cudaStream_t s) {
    const long long n = (long long)B * n_tokens;
    tokens_to_spins_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(B, n_tokens, P, tokens, site_index, spins);
    return cudaGetLastError();
}

cudaError_t fv_launch_free_energy(int B, const float* E, const float* logq, double T, double* out, cudaStream_t s) {
    free_energy_kernel<<<1, 1024, 0, s>>>(B, E, logq, T, out);
    return cudaGetLastError();
}
