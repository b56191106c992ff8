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

// Where the z columns of the design region sit in the caller's 4-D arrays, in 16-byte pieces of the array's element type
// (2 complex64 cells of a field, 4 floats of eps).  Dense region arrays [B,3,nx,ny,nz]: column col = i*ny + j of plane (b,c)
// starts at ((b*3+c)*ncol + col) * col_pitch.  Embedded in a simulation domain [B,3,NXf,NYf,NZf] with the design region at
// (i0,j0,k0) (epsgrad_plan_set_embedding; "|Omega_D"): at (((b*3+c)*NXf + i0+i)*NYf + j0+j)*col_pitch + k0 (pieces).
struct ColumnMap {
    int embedded, ny;
    unsigned col_pitch;                 // pieces per z column of the caller's array
    size_t row_pitch, plane_pitch, base;
    __device__ __forceinline__ size_t plane(int b, int c) const { return ((size_t)b * 3 + c) * plane_pitch + base; }
    __device__ __forceinline__ size_t col(int idx) const
    {
        if (!embedded) return (size_t)idx * col_pitch;
        const int i = idx / ny, j = idx - i * ny;
        return (size_t)i * row_pitch + (size_t)j * col_pitch;
    }
};

// streaming 16-byte load that does not allocate in L1 (fields are read exactly once).
// SPARSE: the access touches only a 64..96-byte window of each 512-byte z column.  By default a
// miss fills the whole 128-byte line from DRAM (measured: 256 B fetched per column for a window
// that straddles a line boundary); the L2::64B prefetch-size qualifier halves that -- 64 B is the
// smallest fill granularity this part honours.
template <bool SPARSE>
__device__ __forceinline__ float4 ld_stream(const float4 *p)
{
    float4 r;
    if (SPARSE)
        asm volatile("ld.global.nc.L1::no_allocate.L2::64B.v4.f32 {%0,%1,%2,%3}, [%4];"
                     : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    else
        asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                     : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}

// Load of a plane that an earlier kernel of the stream produced (CG = false: default caching) or that other CTAs of the SAME
// launch produce (CG = true, the persistent kernel of mega.cuh: L1 is not coherent, so the load goes to L2).
template <bool CG>
__device__ __forceinline__ float ld_plane(const float *p) { return CG ? __ldcg(p) : *p; }
template <bool CG>
__device__ __forceinline__ float2 ld_plane2(const float2 *p) { return CG ? __ldcg(p) : *p; }

// Programmatic dependent launch (sm_90+): a kernel launched with the programmatic-stream-serialization attribute may start
// while the kernel before it on the stream is still running; pdl_wait() blocks until that kernel has completed and its writes
// are visible (a no-op for a normal launch), pdl_launch() lets the NEXT kernel's CTAs be scheduled early (a no-op without a
// dependent).  The kernels of the path call pdl_launch() first and pdl_wait() before they touch anything another kernel
// wrote: launch latency, CTA ramp-up and table staging of a kernel then overlap the tail of its predecessor.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// 1/x on the special-function unit (MUFU.RCP, <= 1 ulp; 1/inf = 0).  The 2-D chain needs ~1e-7
// relative accuracy (tolerances 1e-5 / 1e-4), not IEEE rounding.
__device__ __forceinline__ float fast_rcp(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// Projection + mixing rule of one mask pixel (Eq. (3)/(6) P:L54,L74):
//   t = beta (Phi - eta), rho = (1 + tanh t)/2 = 1/(1 + exp(-2t)), e = eps_clad + (eps_core - eps_clad) rho.
// phi_c is the centred filter output Phi - eta0; eta_r = eta - eta0.  exp(-2t) -> +inf gives rho = 0,
// -> 0 gives rho = 1: no NaN.  |d rho| <= rho (1-rho) * relerr(exp) < 1e-7 with the ex2.approx path
// (DESIGN.md 6.2).
__device__ __forceinline__ float project_mix(float phi_c, float beta, float eta_r, float eps_clad, float deps)
{
    const float t = beta * (phi_c - eta_r);
    const float rho = fast_rcp(1.0f + __expf(-2.0f * t));
    return fmaf(deps, rho, eps_clad);
}

// d rho / d Phi = (beta/2) sech^2 t in the overflow-free form 2 beta a/(1+a)^2, a = exp(-2|t|)
// (the paper's custom tanh derivative rule).
__device__ __forceinline__ float project_slope(float phi_c, float beta, float eta_r)
{
    const float t = beta * (phi_c - eta_r);
    const float a = __expf(-2.0f * fabsf(t));
    const float d = fast_rcp(1.0f + a);
    return 2.0f * beta * a * d * d;
}

// load N consecutive floats from shared memory (N even; 16-byte vectors when N % 4 == 0 and p is 16-byte aligned)
template <int N>
__device__ __forceinline__ void lds_vec(const float *p, float *out)
{
    if (N % 4 == 0) {
#pragma unroll
        for (int q = 0; q < N / 4; ++q) {
            const float4 t = reinterpret_cast<const float4 *>(p)[q];
            out[4 * q] = t.x; out[4 * q + 1] = t.y; out[4 * q + 2] = t.z; out[4 * q + 3] = t.w;
        }
    } else {
#pragma unroll
        for (int q = 0; q < N / 2; ++q) {
            const float2 t = reinterpret_cast<const float2 *>(p)[q];
            out[2 * q] = t.x; out[2 * q + 1] = t.y;
        }
    }
}

struct Normaliser {          // 1/sum_w lookup (S2), DESIGN.md 5.1
    const float *tab;        // conic: [KX*m][KY*m]; separable: x table [KX*m] then y table [KY*m]; plane: [px][plane_py]
    int mx, my, m, T, KX, KY, separable;
    int plane_py;            // > 0: tab is a whole plane of 1/sum_w on the mask, written by k_filter_general (a non-integer number
                             // of cells per control pixel has no phase structure to tabulate); index = pixel coordinate
    // table row / column of mask pixel p = m*a0 + f along x / y
    __device__ __forceinline__ int ix(int a0, int f) const { return border_class(a0, mx, T, KX) * m + f; }
    __device__ __forceinline__ int iy(int b0, int f) const { return border_class(b0, my, T, KY) * m + f; }
    __device__ __forceinline__ int ix_of(int p) const { if (plane_py) return p; const int a0 = p / m; return ix(a0, p - a0 * m); }
    __device__ __forceinline__ int iy_of(int q) const { if (plane_py) return q; const int b0 = q / m; return iy(b0, q - b0 * m); }
    __device__ __forceinline__ float at_index(int i, int j) const
    {
        if (plane_py) return tab[(size_t)i * plane_py + j];
        return separable ? tab[i] * tab[KX * m + j] : tab[i * (KY * m) + j];
    }
    __device__ __forceinline__ float at(int p, int q) const { return at_index(ix_of(p), iy_of(q)); }
};

}  // namespace epsgrad
