// reduce.cuh -- small deterministic reductions of the beta-related outputs (NEXT-2):
//   d F / d beta: eps_hat is differentiable in beta too.  Per mask pixel the projection contributes
//       rhobar d rho/d beta = Phibar (x - eta) / beta,   Phibar = rhobar (beta/2) sech^2 t  (the cotangent the reverse pass forms anyway),
//   so maskgrad.cuh / morph.cuh leave one partial sum per CTA and k_sum_partials adds them in a fixed order.
//   u(beta), the "relative number of gray pixels" (S20: the mean over the mask of 4 rho (1 - rho) = sech^2 t).
// No atomics: the results are bitwise reproducible.
#pragma once
#include "common.cuh"
#include "sizes.cuh"

namespace epsgrad {

// sum of v over the CTA (blockDim.x a multiple of 32, <= 1024); the result is valid in thread 0
__device__ __forceinline__ float block_sum(float v, float *scratch /* >= 32 floats of shared memory */)
{
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    __syncthreads();                                   // scratch may still be in use by an earlier call
    if (lane == 0) scratch[warp] = v;
    __syncthreads();
    float s = 0.f;
    if (warp == 0) {
        s = lane < nw ? scratch[lane] : 0.f;
        for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    }
    return s;
}

// out[b] = scale * (sum_i pa[b*na + i] + sum_i pb[b*nb + i]); grid B, 256 threads; nb may be 0
__global__ void __launch_bounds__(256) k_sum_partials(const float *pa, int na, const float *pb, int nb, float scale, float *out)
{
    __shared__ float scratch[32];
    float v = 0.f;
    for (int i = threadIdx.x; i < na; i += 256) v += pa[(size_t)blockIdx.x * na + i];
    for (int i = threadIdx.x; i < nb; i += 256) v += pb[(size_t)blockIdx.x * nb + i];
    const float s = block_sum(v, scratch);
    if (threadIdx.x == 0) out[blockIdx.x] = scale * s;
}


// partial sums of sech^2(beta (x - eta_r)) over the mask of design blockIdx.y; x: centred input of the last projection
__global__ void __launch_bounds__(UB_THREADS) k_unbinarity(const float *x, size_t n_mask, float beta, float eta_r, float *part)
{
    __shared__ float scratch[32];
    const float *xb = x + (size_t)blockIdx.y * n_mask;
    const size_t base = (size_t)blockIdx.x * (UB_THREADS * UB_PER_THREAD) + threadIdx.x;
    float v = 0.f;
#pragma unroll 4
    for (int k = 0; k < UB_PER_THREAD; ++k) {
        const size_t i = base + (size_t)k * UB_THREADS;
        if (i < n_mask) {
            const float a = __expf(-2.0f * fabsf(beta * (xb[i] - eta_r)));     // 4 rho (1 - rho) = sech^2 t = 4a/(1+a)^2
            const float d = fast_rcp(1.0f + a);
            v += 4.0f * a * d * d;
        }
    }
    const float s = block_sum(v, scratch);
    if (threadIdx.x == 0) part[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = s;
}

}  // namespace epsgrad
