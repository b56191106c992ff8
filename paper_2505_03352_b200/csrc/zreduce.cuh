// zreduce.cuh -- R1 of the reverse pass: Eq. (1) cotangent and its z-reduction.
//   G3 = -2 Re(E_F (.) E_A) = -2 (Re E_F Re E_A - Im E_F Im E_A)           (S10)
//   gbar[x|y][i,j] = sum_k wxy_k G3[c,i,j,k]                (transpose of the z-extrusion)
//   eps_zz,k = 1/(wz_k/eps2d_z + (1-wz_k)/eps_clad): its derivative w.r.t. eps2d_z is 1 on
//   full cells (wz_k = 1) and depends on eps2d_z only on the (at most two) fractional
//   face cells, so the z component is reduced to three planes -- full cells, lower face,
//   upper face -- and the 2-D reverse kernel applies the face factors.  This keeps the
//   field stream independent of the 2-D chain.
// Only the 16-byte chunks (2 complex64 cells) of a z column that hold slab cells are read
// ("|Omega_D"; d eps/dC = 0 elsewhere); `dense` plans read every chunk.  L lanes
// (a power of two) share a column and reduce with xor-shuffles; each thread keeps
// ZR_UNROLL columns in flight so that 2*ZR_UNROLL 16-byte loads are issued before use.  Consecutive
// lane groups take consecutive columns, so one warp instruction covers 32/L neighbouring columns.
// SPARSE windows (<= 128 B of a column) use 64-byte L2 fills (common.cuh ld_stream).
#pragma once
#include "common.cuh"

namespace epsgrad {

constexpr int ZR_THREADS = 256, ZR_MAX_PAIRS = 8;
constexpr int ZR_UNROLL_SPARSE = 2, ZR_UNROLL_DENSE = 4;   // columns in flight per thread (swept on B200: profiles/r1b_notes.md)

struct ZredParams {
    const float4 *ef[ZR_MAX_PAIRS];
    const float4 *ea[ZR_MAX_PAIRS];
    float *gbar;           // [B,5,ncol]
    const float *zw;       // [5][nz]: wxy, wz, z-full indicator, z-lower-face indicator, z-upper-face indicator
    int n_pairs, accumulate;
    int ncol, nz;
    int ch0[2], nch[2], L[2];   // chunk window (chunk = 2 cells) and lanes per column for {x,y} and {z}
};

// One block of columns (index bx) of component c of design b.
template <int ZR_UNROLL, bool SPARSE>
__device__ __forceinline__ void zreduce_block(const ZredParams &P, int bx, int c, int b)
{
    const int grp = c == 2;
    const int L = P.L[grp], ch0 = P.ch0[grp], nch = P.nch[grp];
    const int tid = threadIdx.x;
    const int l = tid & (L - 1), g = tid / L, GPB = ZR_THREADS / L;
    const int nzc = P.nz >> 1;                       // chunks per column
    const size_t plane = ((size_t)b * 3 + c) * P.ncol;

    // thread's columns: colbase + u*GPB (consecutive lane groups take consecutive columns)
    const int colbase = bx * (ZR_UNROLL * GPB) + g;
    if (colbase - g >= P.ncol) return;               // whole block past the end (uniform)
    bool live[ZR_UNROLL];
#pragma unroll
    for (int u = 0; u < ZR_UNROLL; ++u) live[u] = colbase + u * GPB < P.ncol;
    const int ustride = GPB * nzc;                   // float4 stride between a thread's columns

    float acc[ZR_UNROLL][3];
#pragma unroll
    for (int u = 0; u < ZR_UNROLL; ++u) acc[u][0] = acc[u][1] = acc[u][2] = 0.0f;

    for (int ch = l; ch < nch; ch += L) {
        const int k = 2 * (ch0 + ch);
        float w[3][2];
        if (grp == 0) {
            w[0][0] = P.zw[k]; w[0][1] = P.zw[k + 1];
            w[1][0] = w[1][1] = w[2][0] = w[2][1] = 0.0f;
        } else {
#pragma unroll
            for (int o = 0; o < 3; ++o) { w[o][0] = P.zw[(2 + o) * P.nz + k]; w[o][1] = P.zw[(2 + o) * P.nz + k + 1]; }
        }
        const size_t off0 = (plane + colbase) * nzc + ch0 + ch;
        for (int p = 0; p < P.n_pairs; ++p) {
            const float4 *pf = P.ef[p] + off0, *pa = P.ea[p] + off0;
            float4 f[ZR_UNROLL], a[ZR_UNROLL];
#pragma unroll
            for (int u = 0; u < ZR_UNROLL; ++u) {
                if (live[u]) {
                    f[u] = ld_stream<SPARSE>(pf + u * ustride);
                    a[u] = ld_stream<SPARSE>(pa + u * ustride);
                } else {
                    f[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                    a[u] = f[u];
                }
            }
#pragma unroll
            for (int u = 0; u < ZR_UNROLL; ++u) {
                const float g0 = -2.0f * (f[u].x * a[u].x - f[u].y * a[u].y);
                const float g1 = -2.0f * (f[u].z * a[u].z - f[u].w * a[u].w);
                acc[u][0] = fmaf(w[0][0], g0, fmaf(w[0][1], g1, acc[u][0]));
                if (grp) {
                    acc[u][1] = fmaf(w[1][0], g0, fmaf(w[1][1], g1, acc[u][1]));
                    acc[u][2] = fmaf(w[2][0], g0, fmaf(w[2][1], g1, acc[u][2]));
                }
            }
        }
    }
    const int nout = grp ? 3 : 1;
#pragma unroll
    for (int u = 0; u < ZR_UNROLL; ++u)
        for (int o = 0; o < nout; ++o) {
            float v = acc[u][o];
            for (int off = L >> 1; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
            acc[u][o] = v;
        }
    if (l != 0) return;
#pragma unroll
    for (int u = 0; u < ZR_UNROLL; ++u) {
        if (!live[u]) continue;
        for (int o = 0; o < nout; ++o) {
            float *dst = P.gbar + ((size_t)b * 5 + (grp ? 2 + o : c)) * P.ncol + colbase + u * GPB;
            *dst = P.accumulate ? *dst + acc[u][o] : acc[u][o];
        }
    }
}

// grid (blocks over columns, 3*B)
template <int ZR_UNROLL, bool SPARSE>
__global__ void __launch_bounds__(ZR_THREADS, 4) k_zreduce(const ZredParams P)
{
    zreduce_block<ZR_UNROLL, SPARSE>(P, blockIdx.x, blockIdx.y % 3, blockIdx.y / 3);
}

}  // namespace epsgrad
