// common.cuh -- shared device helpers of the epsgrad CUDA path (sm_100a).
// Product code: shares nothing with oracle/.  Notation follows the paper (arxiv
// 2505.03352) and DESIGN.md: u = Yee cells per control pixel, s = mask pixels per Yee
// cell, m = u*s mask pixels per control pixel, T = half-range of filter taps in control
// pixels, NT = 2T+1.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace epsgrad {

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

// Border class of control index a0 along an axis with M nodes: the set of
// in-range filter taps, hence the normaliser of Eq. (2) (S2), depends on a0 only within T
// nodes of either end.  K = 2T+1 classes when M >= 2T+1, else K = M and class = a0.
__device__ __forceinline__ int border_class(int a0, int M, int T, int K)
{
    if (K == M) return a0;
    if (a0 < T) return a0;
    const int d = M - 1 - a0;
    return d < T ? 2 * T - d : T;
}

// streaming 16-byte load that does not allocate in L1 (fields are read exactly once)
__device__ __forceinline__ float4 ld_stream(const float4 *p)
{
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}

// Projection + mixing rule of one mask pixel (Eq. (3)/(6) P:L54,L74):
//   t = beta (Phi - eta), rho = (1 + tanh t)/2, e = eps_clad + (eps_core - eps_clad) rho.
// phi_c is the centred filter output Phi - eta0; eta_r = eta - eta0.
__device__ __forceinline__ float project_mix(float phi_c, float beta, float eta_r, float eps_clad, float deps)
{
    const float t = beta * (phi_c - eta_r);
    const float rho = 0.5f * (1.0f + tanhf(t));
    return fmaf(deps, rho, eps_clad);
}

// d rho / d Phi = (beta/2) sech^2 t in the overflow-free form 2 beta a/(1+a)^2, a = exp(-2|t|)
// (the paper's custom tanh derivative rule).
__device__ __forceinline__ float project_slope(float phi_c, float beta, float eta_r)
{
    const float t = beta * (phi_c - eta_r);
    const float a = expf(-2.0f * fabsf(t));
    const float d = 1.0f + a;
    return 2.0f * beta * a / (d * d);
}

struct Normaliser {          // 1/sum_w lookup (S2), DESIGN.md 5.1
    const float *tab;        // conic: [KX*m][KY*m]; separable: x table [KX*m] then y table [KY*m]
    int mx, my, m, T, KX, KY, separable;
    __device__ __forceinline__ float at(int p, int q) const
    {
        const int a0 = p / m, fx = p - a0 * m, b0 = q / m, fy = q - b0 * m;
        const int ix = border_class(a0, mx, T, KX) * m + fx;
        const int iy = border_class(b0, my, T, KY) * m + fy;
        return separable ? tab[ix] * tab[KX * m + iy] : tab[ix * (KY * m) + iy];
    }
};

}  // namespace epsgrad
