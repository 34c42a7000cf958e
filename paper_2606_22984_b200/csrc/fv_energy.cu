// fv_energy.cu -- batched Ising energies and the F_q reduction for sm_100a.
//   EA lattices: E_b = -sum_bonds J_ij s_i s_j, CSR gather-reduce      (Eq. 8)
//   dense SK   : E_b = -sum_{i<j} J_ij s_i s_j                          (Eq. 6)
//   F_q        : mean_b(E_b + T log q_b) and its std                    (Eq. 5)
// All reductions use a fixed tree (shuffle, then shared memory) => bit-reproducible.
#include "fv_internal.h"

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
    if (threadIdx.x == 0) { out[0] = mean; out[1] = sqrt(var); }
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
    const size_t smem = (size_t)8 * N;
    if (smem > 200 * 1024) return cudaErrorInvalidValue;
    if (smem > 48 * 1024) cudaFuncSetAttribute(energy_dense_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    energy_dense_kernel<<<(B + 7) / 8, 256, smem, s>>>(B, N, spins, J, E);
    return cudaGetLastError();
}

cudaError_t fv_launch_free_energy(int B, const float* E, const float* logq, double T, double* out, cudaStream_t s) {
    free_energy_kernel<<<1, 1024, 0, s>>>(B, E, logq, T, out);
    return cudaGetLastError();
}
