// forward.cuh -- steps 3-7 of the chain fused in one tile kernel:
//   projection + mixing (Eq. (3)/(6)) -> cell averages on the half-cell
//   shifted footprints (Eq. (8)) -> Sobel normals -> Eq. (7)
//    -> z-extrusion with fractional faces (S7,S8), streamed to HBM.
// One CTA owns TI x TJ Yee cells: it reads the (L2-resident) centred filter output Phi'
// for its tile plus a one-cell halo, keeps every 2-D intermediate in shared memory and
// then writes its 3 x TI x TJ z-columns with 16-byte streaming stores.  The store stream
// (12 B per Yee cell) is the only HBM traffic that matters; the 2-D work of other
// resident CTAs overlaps it.
#pragma once
#include "common.cuh"

namespace epsgrad {

struct FwdParams {
    const float *phi;      // [B,px,py]
    float *eps;            // [B,3,nx,ny,nz] or nullptr
    float *eps2d;          // [B,3,nx,ny] or nullptr (stage tap)
    const float *zw;       // [7][nz] z tables (epsgrad.cu): wxy, wz, z-full, z-lower-face, z-upper-face indicators,
                           //          eps_clad (1 - wxy), eps_clad [wz == 0]
    int nx, ny, nz, px, py, s;
    float beta, eta_r, eps_clad, deps, delta;
    float w_lo, w_hi;      // fractional z-face weights of eps_zz (0 if that face cell is absent)
};

constexpr int FWD_TI = 16, FWD_TJ = 16, FWD_THREADS = 256;

__host__ __device__ inline size_t fwd_smem_floats(int s, int nz)
{
    const int CI = FWD_TI + 2, CJ = FWD_TJ + 2;
    const int MP = s * CI + s / 2, MQ = s * CJ + s / 2;
    return (size_t)2 * MP * MQ + 4 * CI * CJ + 5 * FWD_TI * FWD_TJ + 7 * (size_t)nz;
}

// One tile (bx, by) of design bz.  S > 0: compile-time subpixel count (index divisions fold to shifts);
// S = 0: runtime P.s.  sm: fwd_smem_floats(s, nz) floats of shared memory.
template <int S>
__device__ __forceinline__ void forward_tile(const FwdParams &P, float *sm, int bx, int by, int bz)
{
    constexpr int TI = FWD_TI, TJ = FWD_TJ, NTH = FWD_THREADS;
    constexpr int CI = TI + 2, CJ = TJ + 2;
    const int s = S > 0 ? S : P.s, hs = s >> 1;
    const int MP = s * CI + hs, MQ = s * CJ + hs;
    float *e_s = sm;
    float *r_s = e_s + MP * MQ;
    float *Ax = r_s + MP * MQ;
    float *Hx = Ax + CI * CJ;
    float *Ay = Hx + CI * CJ;
    float *Hy = Ay + CI * CJ;
    float *e2 = Hy + CI * CJ;          // [5][TI*TJ]: eps2d_x, eps2d_y, eps2d_z, eps_zz on the lower / upper face cell
    float *zw = e2 + 5 * TI * TJ;      // [7][nz]

    const int tid = threadIdx.x;
    const int i0 = by * TI, j0 = bx * TJ, b = bz;
    const int nx = P.nx, ny = P.ny, nz = P.nz;
    const float inv_s2 = 1.0f / (float)(s * s);

    for (int k = tid; k < 7 * nz; k += NTH) zw[k] = P.zw[k];

    // ---- stage 1: mask tile (replicate outside the region, S5): e and r = 1/e
    {
        const float *phib = P.phi + (size_t)b * P.px * P.py;
        const int p_base = s * (i0 - 1), q_base = s * (j0 - 1);
        for (int i = tid; i < MP * MQ; i += NTH) {
            const int lp = i / MQ, lq = i - lp * MQ;
            const int p = clampi(p_base + lp, 0, P.px - 1), q = clampi(q_base + lq, 0, P.py - 1);
            const float e = project_mix(phib[p * P.py + q], P.beta, P.eta_r, P.eps_clad, P.deps);
            e_s[i] = e;
            r_s[i] = fast_rcp(e);
        }
    }
    __syncthreads();

    // ---- stage 2: <e>, <1/e> on the E_x and E_y footprints for the tile + 1-cell halo
    for (int i = tid; i < CI * CJ; i += NTH) {
        const int ci = i / CJ, cj = i - ci * CJ;
        const int lp0 = s * ci, lq0 = s * cj;
        float ax = 0.f, hx = 0.f, ay = 0.f, hy = 0.f;
        for (int a = 0; a < s; ++a)
            for (int bb = 0; bb < s; ++bb) {
                const int ix = (lp0 + hs + a) * MQ + lq0 + bb;       // E_x: half a cell toward +x
                const int iy = (lp0 + a) * MQ + lq0 + hs + bb;       // E_y: half a cell toward +y
                ax += e_s[ix]; hx += r_s[ix];
                ay += e_s[iy]; hy += r_s[iy];
            }
        Ax[i] = ax * inv_s2; Hx[i] = hx * inv_s2;
        Ay[i] = ay * inv_s2; Hy[i] = hy * inv_s2;
    }
    __syncthreads();

    // ---- stage 3: Sobel normals of D_c = (A_c - eps_clad)/deps, Eq. (7); eps2d_z = <e>_z
    const float inv_deps = 1.0f / P.deps;
    const bool inner = i0 >= 1 && j0 >= 1 && i0 + TI <= nx - 1 && j0 + TJ <= ny - 1;   // 1-cell ring inside the region
    for (int it = tid; it < TI * TJ; it += NTH) {
        const int ii = it / TJ, jj = it - ii * TJ;
        const int i = i0 + ii, j = j0 + jj;
        if (i >= nx || j >= ny) continue;
        float out[3];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const float *A = c == 0 ? Ax : Ay, *H = c == 0 ? Hx : Hy;
            float gx, gy;
            if (inner) {
                const float *q1 = A + (ii + 1) * CJ + jj + 1, *q0 = q1 - CJ, *q2 = q1 + CJ;
                const float a00 = q0[-1], a01 = q0[0], a02 = q0[1], a10 = q1[-1], a12 = q1[1];
                const float a20 = q2[-1], a21 = q2[0], a22 = q2[1];
                gx = ((a20 - a00) + 2.0f * (a21 - a01) + (a22 - a02)) * 0.125f;
                gy = ((a02 - a00) + 2.0f * (a12 - a10) + (a22 - a20)) * 0.125f;
            } else {
                gx = 0.f; gy = 0.f;
#pragma unroll
                for (int di = -1; di <= 1; ++di)
#pragma unroll
                    for (int dj = -1; dj <= 1; ++dj) {
                        const int ni = clampi(i + di, 0, nx - 1) - (i0 - 1);
                        const int nj = clampi(j + dj, 0, ny - 1) - (j0 - 1);
                        const float d = A[ni * CJ + nj];
                        gx = fmaf((float)(di * (2 - (dj < 0 ? -dj : dj))) * 0.125f, d, gx);
                        gy = fmaf((float)(dj * (2 - (di < 0 ? -di : di))) * 0.125f, d, gy);
                    }
            }
            gx *= inv_deps; gy *= inv_deps;
            const float gc = c == 0 ? gx : gy;
            const float n2 = gc * gc * fast_rcp(gx * gx + gy * gy + P.delta);
            const int ic = (ii + 1) * CJ + jj + 1;
            out[c] = fast_rcp(n2 * H[ic] + (1.0f - n2) * fast_rcp(A[ic]));
        }
        {
            float az = 0.f;
            const int lp0 = s * (ii + 1), lq0 = s * (jj + 1);
            for (int a = 0; a < s; ++a)
                for (int bb = 0; bb < s; ++bb) az += e_s[(lp0 + a) * MQ + lq0 + bb];
            out[2] = az * inv_s2;
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            e2[c * TI * TJ + it] = out[c];
            if (P.eps2d) P.eps2d[(((size_t)b * 3 + c) * nx + i) * ny + j] = out[c];
        }
        // Eq. (7) with n = z_hat on the (at most two) fractional face cells of E_z (S7): once per column
        const float inv_ec = 1.0f / P.eps_clad;
        const float rz = fast_rcp(out[2]);
        e2[3 * TI * TJ + it] = P.w_lo > 0.f ? fast_rcp(P.w_lo * rz + (1.0f - P.w_lo) * inv_ec) : 0.f;
        e2[4 * TI * TJ + it] = P.w_hi > 0.f ? fast_rcp(P.w_hi * rz + (1.0f - P.w_hi) * inv_ec) : 0.f;
    }
    if (!P.eps) return;
    __syncthreads();

    // ---- stage 4: z-extrusion, 16-byte streaming stores.  Every output is affine in the staged per-column values:
    //   eps_cc[k] = eps_clad (1 - wxy_k) + wxy_k eps2d_c          (c = x, y)
    //   eps_zz[k] = eps_clad [wz_k = 0] + [wz_k = 1] eps2d_z + [k = lower face] v_lo + [k = upper face] v_hi
    const int TIv = min(TI, nx - i0), TJv = min(TJ, ny - j0);
    const int nz4 = nz >> 2;
    const float *w_xy = zw, *b_xy = zw + 5 * nz, *b_z = zw + 6 * nz, *i_f = zw + 2 * nz, *i_l = zw + 3 * nz, *i_h = zw + 4 * nz;
    if (NTH % nz4 == 0) {
        // a thread keeps its 4 z cells for the whole tile: weights live in registers
        const int kc = tid % nz4, k = kc << 2, cstep = NTH / nz4;
        float wx[4], bx[4], bz[4], zf[4], zl[4], zh[4];
#pragma unroll
        for (int x = 0; x < 4; ++x) {
            wx[x] = w_xy[k + x]; bx[x] = b_xy[k + x]; bz[x] = b_z[k + x];
            zf[x] = i_f[k + x]; zl[x] = i_l[k + x]; zh[x] = i_h[k + x];
        }
        for (int c = 0; c < 3; ++c) {
            float *base = P.eps + ((((size_t)b * 3 + c) * nx + i0) * ny + j0) * nz + k;   // tile-relative offsets fit 32 bits
            const float *vc = e2 + c * TI * TJ;
            const int row_stride = ny * nz;
            for (int cell = tid / nz4; cell < TIv * TJ; cell += cstep) {
                const int ii = cell / TJ, jj = cell - ii * TJ;
                if (jj >= TJv) continue;
                const float v = vc[cell];
                float4 o;
                if (c < 2) {
                    o.x = fmaf(wx[0], v, bx[0]); o.y = fmaf(wx[1], v, bx[1]);
                    o.z = fmaf(wx[2], v, bx[2]); o.w = fmaf(wx[3], v, bx[3]);
                } else {
                    const float vl = e2[3 * TI * TJ + cell], vh = e2[4 * TI * TJ + cell];
                    o.x = fmaf(zf[0], v, fmaf(zl[0], vl, fmaf(zh[0], vh, bz[0])));
                    o.y = fmaf(zf[1], v, fmaf(zl[1], vl, fmaf(zh[1], vh, bz[1])));
                    o.z = fmaf(zf[2], v, fmaf(zl[2], vl, fmaf(zh[2], vh, bz[2])));
                    o.w = fmaf(zf[3], v, fmaf(zl[3], vl, fmaf(zh[3], vh, bz[3])));
                }
                __stcs(reinterpret_cast<float4 *>(base + (ii * row_stride + jj * nz)), o);
            }
        }
    } else {
        for (int c = 0; c < 3; ++c) {
            float *base = P.eps + ((((size_t)b * 3 + c) * nx + i0) * ny + j0) * nz;
            const float *vc = e2 + c * TI * TJ;
            for (int f = tid; f < TIv * TJ * nz4; f += NTH) {
                const int cell = f / nz4, k = (f - cell * nz4) << 2;
                const int ii = cell / TJ, jj = cell - ii * TJ;
                if (jj >= TJv) continue;
                const float v = vc[cell], vl = e2[3 * TI * TJ + cell], vh = e2[4 * TI * TJ + cell];
                float o[4];
#pragma unroll
                for (int x = 0; x < 4; ++x)
                    o[x] = c < 2 ? fmaf(w_xy[k + x], v, b_xy[k + x])
                                 : fmaf(i_f[k + x], v, fmaf(i_l[k + x], vl, fmaf(i_h[k + x], vh, b_z[k + x])));
                __stcs(reinterpret_cast<float4 *>(base + ((size_t)ii * ny + jj) * nz + k), make_float4(o[0], o[1], o[2], o[3]));
            }
        }
    }
}

// grid (ceil(ny/TJ), ceil(nx/TI), B)
template <int S>
__global__ void __launch_bounds__(FWD_THREADS) k_forward(const FwdParams P)
{
    extern __shared__ __align__(16) float sm[];
    forward_tile<S>(P, sm, blockIdx.x, blockIdx.y, blockIdx.z);
}

}  // namespace epsgrad
