// extrude.cuh -- F6: z-extrusion of the 2-D stage to the slab [z_lo, z_hi] with fractional faces (S7, S8).
// Pure store stream: 12 B per Yee cell written with 16-byte streaming stores, 20 B per Yee column read (L2-resident
// planes left by fwd2d.cuh).  Every output is affine in the per-column values:
//   eps_cc[k] = eps_clad (1 - wxy_k) + wxy_k eps2d_c                                         (c = x, y)
//   eps_zz[k] = eps_clad [wz_k = 0] + [wz_k = 1] eps2d_z + [k = lower face] v_lo + [k = upper face] v_hi
// where v_lo, v_hi are Eq. (7) with n = z_hat on the face cells (computed once per column by fwd2d).
// nz/4 threads share a column, each keeping its four z cells and their table entries in registers for the whole CTA;
// a warp store covers 32/(nz/4) neighbouring columns = 512 contiguous bytes; EX_UNROLL columns per thread are in
// flight so that the plane loads of the next columns overlap the stores of the current ones.
#pragma once
#include "common.cuh"

namespace epsgrad {

constexpr int EX_THREADS = 256, EX_UNROLL = 4, EX_PASSES = 2;   // a CTA owns (EX_THREADS / (nz/4)) * EX_UNROLL * EX_PASSES columns

struct ExtrudeParams {
    const float *e2d;      // [B,5,ncol]: eps2d_x, eps2d_y, eps2d_z, eps_zz lower face, eps_zz upper face
    float *eps;            // [B,3,ncol,nz]
    const float *zw;       // [7][nz] z tables (epsgrad.cu)
    int ncol, nz;
};

__host__ __device__ inline int extrude_cols_per_cta(int nz)
{
    const int nz4 = nz >> 2;
    return EX_THREADS % nz4 == 0 ? (EX_THREADS / nz4) * EX_UNROLL * EX_PASSES : 64;
}

// grid (ceil(ncol / extrude_cols_per_cta), B)
__global__ void __launch_bounds__(EX_THREADS) k_extrude(const __grid_constant__ ExtrudeParams P)
{
    const int tid = threadIdx.x, b = blockIdx.y, nz = P.nz, nz4 = nz >> 2, ncol = P.ncol;
    const float *w_xy = P.zw, *b_xy = P.zw + 5 * nz, *b_z = P.zw + 6 * nz, *i_f = P.zw + 2 * nz, *i_l = P.zw + 3 * nz, *i_h = P.zw + 4 * nz;
    const float *ed = P.e2d + (size_t)b * 5 * ncol;
    float *out = P.eps + (size_t)b * 3 * ncol * nz;
    const int cpc = extrude_cols_per_cta(nz), colb = blockIdx.x * cpc;
    if (EX_THREADS % nz4 == 0) {
        const int k = (tid % nz4) << 2, cq = tid / nz4, cpp = EX_THREADS / nz4;
        float wx[4], bx[4], bz[4], zf[4], zl[4], zh[4];
#pragma unroll
        for (int x = 0; x < 4; ++x) {
            wx[x] = w_xy[k + x]; bx[x] = b_xy[k + x]; bz[x] = b_z[k + x];
            zf[x] = i_f[k + x]; zl[x] = i_l[k + x]; zh[x] = i_h[k + x];
        }
        for (int pass = 0; pass < EX_PASSES; ++pass) {
            const int col0 = colb + pass * cpp * EX_UNROLL + cq;
            float v[EX_UNROLL][5];
#pragma unroll
            for (int u = 0; u < EX_UNROLL; ++u) {
                const int col = col0 + u * cpp;
                if (col < ncol) {
#pragma unroll
                    for (int o = 0; o < 5; ++o) v[u][o] = __ldg(ed + (size_t)o * ncol + col);
                }
            }
#pragma unroll
            for (int u = 0; u < EX_UNROLL; ++u) {
                const int col = col0 + u * cpp;
                if (col < ncol) {
                    float4 *dst = reinterpret_cast<float4 *>(out + (size_t)col * nz + k);
                    const size_t cstride = (size_t)ncol * nz4;        // float4 stride between component planes
                    float4 o;
                    o.x = fmaf(wx[0], v[u][0], bx[0]); o.y = fmaf(wx[1], v[u][0], bx[1]);
                    o.z = fmaf(wx[2], v[u][0], bx[2]); o.w = fmaf(wx[3], v[u][0], bx[3]);
                    __stcs(dst, o);
                    o.x = fmaf(wx[0], v[u][1], bx[0]); o.y = fmaf(wx[1], v[u][1], bx[1]);
                    o.z = fmaf(wx[2], v[u][1], bx[2]); o.w = fmaf(wx[3], v[u][1], bx[3]);
                    __stcs(dst + cstride, o);
                    o.x = fmaf(zf[0], v[u][2], fmaf(zl[0], v[u][3], fmaf(zh[0], v[u][4], bz[0])));
                    o.y = fmaf(zf[1], v[u][2], fmaf(zl[1], v[u][3], fmaf(zh[1], v[u][4], bz[1])));
                    o.z = fmaf(zf[2], v[u][2], fmaf(zl[2], v[u][3], fmaf(zh[2], v[u][4], bz[2])));
                    o.w = fmaf(zf[3], v[u][2], fmaf(zl[3], v[u][3], fmaf(zh[3], v[u][4], bz[3])));
                    __stcs(dst + 2 * cstride, o);
                }
            }
        }
    } else {
        // nz/4 does not divide the CTA: flat loop over the 16-byte pieces of the CTA's columns
        const int ncb = min(cpc, ncol - colb);
        for (int c = 0; c < 3; ++c)
            for (int f = tid; f < ncb * nz4; f += EX_THREADS) {
                const int lc = f / nz4, k = (f - lc * nz4) << 2, col = colb + lc;
                const float v = ed[(size_t)c * ncol + col], vl = ed[(size_t)3 * ncol + col], vh = ed[(size_t)4 * ncol + col];
                float o[4];
#pragma unroll
                for (int x = 0; x < 4; ++x)
                    o[x] = c < 2 ? fmaf(w_xy[k + x], v, b_xy[k + x])
                                 : fmaf(i_f[k + x], v, fmaf(i_l[k + x], vl, fmaf(i_h[k + x], vh, b_z[k + x])));
                __stcs(reinterpret_cast<float4 *>(out + ((size_t)c * ncol + col) * nz + k), make_float4(o[0], o[1], o[2], o[3]));
            }
    }
}

}  // namespace epsgrad
