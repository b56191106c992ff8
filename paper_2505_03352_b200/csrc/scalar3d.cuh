// scalar3d.cuh -- the two 3-D steps for z columns that the 16-byte paths cannot address (nz not a multiple of 4: a column of
// eps is then not a whole number of 16-byte pieces, and for odd nz a field column does not start on a 16-byte boundary):
//   k_extrude_scalar  F6, one thread per Yee cell, 4-byte stores (extrude.cuh has the formulas: same affine forms);
//   k_zreduce_scalar  R1, one thread per z column, 8-byte loads of the slab cells (zreduce.cuh: same product, same planes).
// Coverage paths for odd grids (region-sized or x-slab arrays, no embedding); every BASELINE config takes the vector paths.
#pragma once
#include "common.cuh"
#include "zreduce.cuh"

namespace epsgrad {

constexpr int SC_THREADS = 256;

struct ExtrudeScalarParams {
    const float *e2d;      // [B,5,pstride] (offset to the slab's first column already applied)
    float *eps;            // [B,3,ncol,nz]
    const float *zw;       // [7][nz]
    int ncol, nz, pstride;
};

// grid (ceil(ncol*nz / SC_THREADS), 3, B)
__global__ void __launch_bounds__(SC_THREADS) k_extrude_scalar(const ExtrudeScalarParams P)
{
    const size_t n = (size_t)P.ncol * P.nz, i = (size_t)blockIdx.x * SC_THREADS + threadIdx.x;
    if (i >= n) return;
    const int c = blockIdx.y, b = blockIdx.z, nz = P.nz;
    const int col = (int)(i / nz), k = (int)(i - (size_t)col * nz);
    const float *ed = P.e2d + (size_t)b * 5 * P.pstride + col;
    float o;
    if (c < 2) o = fmaf(__ldg(P.zw + k), ed[(size_t)c * P.pstride], __ldg(P.zw + 5 * nz + k));
    else o = fmaf(__ldg(P.zw + 2 * nz + k), ed[(size_t)2 * P.pstride],
                  fmaf(__ldg(P.zw + 3 * nz + k), ed[(size_t)3 * P.pstride], fmaf(__ldg(P.zw + 4 * nz + k), ed[(size_t)4 * P.pstride], __ldg(P.zw + 6 * nz + k))));
    P.eps[((size_t)b * 3 + c) * n + i] = o;
}

struct ZredScalarParams {
    const float2 *ef[ZR_MAX_PAIRS];
    const float2 *ea[ZR_MAX_PAIRS];
    float *gbar;           // [B,5,pstride] (offset to the slab's first column already applied)
    const float *zw;       // [7][nz]
    int n_pairs, accumulate;
    int ncol, nz, pstride;
    int k0[2], k1[2];      // first / one-past-last slab cell for {x,y} and {z}
};

// grid (ceil(ncol / SC_THREADS), 3, B)
__global__ void __launch_bounds__(SC_THREADS) k_zreduce_scalar(const ZredScalarParams P)
{
    const int col = blockIdx.x * SC_THREADS + threadIdx.x;
    if (col >= P.ncol) return;
    const int c = blockIdx.y, b = blockIdx.z, grp = c == 2, nz = P.nz;
    const size_t base = (((size_t)b * 3 + c) * P.ncol + col) * nz;
    float acc[3] = {0.f, 0.f, 0.f};
    for (int p = 0; p < P.n_pairs; ++p)
        for (int k = P.k0[grp]; k < P.k1[grp]; ++k) {
            const float2 f = P.ef[p][base + k], a = P.ea[p][base + k];
            const float g = -2.0f * (f.x * a.x - f.y * a.y);                // Eq. (1): -2 Re(E_F E_A), plain product (S10)
            if (grp == 0) acc[0] = fmaf(__ldg(P.zw + k), g, acc[0]);
            else {
#pragma unroll
                for (int o = 0; o < 3; ++o) acc[o] = fmaf(__ldg(P.zw + (2 + o) * nz + k), g, acc[o]);
            }
        }
    float *dst = P.gbar + (size_t)b * 5 * P.pstride + col;
    const int nout = grp ? 3 : 1;
    for (int o = 0; o < nout; ++o) {
        float *d = dst + (size_t)(grp ? 2 + o : c) * P.pstride;
        *d = P.accumulate ? *d + acc[o] : acc[o];
    }
}

}  // namespace epsgrad
