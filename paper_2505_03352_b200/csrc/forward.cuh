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
    const float *zw;       // [2][nz]: wxy_k, wz_k (overlaps of the z footprints with the slab)
    int nx, ny, nz, px, py, s;
    float beta, eta_r, eps_clad, deps, delta;
};

constexpr int FWD_TI = 16, FWD_TJ = 16, FWD_THREADS = 256;

__host__ __device__ inline size_t fwd_smem_floats(int s, int nz)
{
    const int CI = FWD_TI + 2, CJ = FWD_TJ + 2;
    const int MP = s * CI + s / 2, MQ = s * CJ + s / 2;
    return (size_t)2 * MP * MQ + 4 * CI * CJ + 3 * FWD_TI * FWD_TJ + 2 * (size_t)nz;
}

// grid (ceil(ny/TJ), ceil(nx/TI), B)
__global__ void __launch_bounds__(FWD_THREADS) k_forward(const FwdParams P)
{
    extern __shared__ __align__(16) float sm[];
    constexpr int TI = FWD_TI, TJ = FWD_TJ, NTH = FWD_THREADS;
    constexpr int CI = TI + 2, CJ = TJ + 2;
    const int s = P.s, hs = s >> 1;
    const int MP = s * CI + hs, MQ = s * CJ + hs;
    float *e_s = sm;
    float *r_s = e_s + MP * MQ;
    float *Ax = r_s + MP * MQ;
    float *Hx = Ax + CI * CJ;
    float *Ay = Hx + CI * CJ;
    float *Hy = Ay + CI * CJ;
    float *e2 = Hy + CI * CJ;          // [3][TI*TJ]
    float *zw = e2 + 3 * TI * TJ;      // [2][nz]

    const int tid = threadIdx.x;
    const int i0 = blockIdx.y * TI, j0 = blockIdx.x * TJ, b = blockIdx.z;
    const int nx = P.nx, ny = P.ny, nz = P.nz;
    const float inv_s2 = 1.0f / (float)(s * s);

    for (int k = tid; k < 2 * nz; k += NTH) zw[k] = P.zw[k];

    // ---- stage 1: mask tile (replicate outside the region, S5): e and r = 1/e
    {
        const float *phib = P.phi + (size_t)b * P.px * P.py;
        const int p_base = s * (i0 - 1), q_base = s * (j0 - 1);
        for (int i = tid; i < MP * MQ; i += NTH) {
            const int lp = i / MQ, lq = i - lp * MQ;
            const int p = clampi(p_base + lp, 0, P.px - 1), q = clampi(q_base + lq, 0, P.py - 1);
            const float e = project_mix(phib[(size_t)p * P.py + q], P.beta, P.eta_r, P.eps_clad, P.deps);
            e_s[i] = e;
            r_s[i] = 1.0f / e;
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
    for (int it = tid; it < TI * TJ; it += NTH) {
        const int ii = it / TJ, jj = it - ii * TJ;
        const int i = i0 + ii, j = j0 + jj;
        if (i >= nx || j >= ny) continue;
        float out[3];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const float *A = c == 0 ? Ax : Ay, *H = c == 0 ? Hx : Hy;
            float gx = 0.f, gy = 0.f;
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
            gx *= inv_deps; gy *= inv_deps;
            const float gc = c == 0 ? gx : gy;
            const float n2 = gc * gc / (gx * gx + gy * gy + P.delta);
            const int ic = (ii + 1) * CJ + jj + 1;
            out[c] = 1.0f / (n2 * H[ic] + (1.0f - n2) / A[ic]);
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
    }
    if (!P.eps) return;
    __syncthreads();

    // ---- stage 4: z-extrusion, 16-byte streaming stores; a (c,i) row of the tile is contiguous
    const int TIv = min(TI, nx - i0), TJv = min(TJ, ny - j0);
    const int nz4 = nz >> 2, n4 = TJv * nz4;
    const float ec = P.eps_clad, inv_ec = 1.0f / P.eps_clad;
    for (int r = 0; r < 3 * TIv; ++r) {
        const int c = r / TIv, ii = r - c * TIv;
        float4 *dst = reinterpret_cast<float4 *>(P.eps + ((((size_t)b * 3 + c) * nx + i0 + ii) * ny + j0) * nz);
        const float *vrow = e2 + c * TI * TJ + ii * TJ;
        for (int f = tid; f < n4; f += NTH) {
            const int jj = f / nz4, k = (f - jj * nz4) << 2;
            const float v = vrow[jj];
            float o[4];
            if (c < 2) {
                const float dv = v - ec;
#pragma unroll
                for (int x = 0; x < 4; ++x) o[x] = fmaf(zw[k + x], dv, ec);
            } else {
#pragma unroll
                for (int x = 0; x < 4; ++x) {
                    const float w = zw[nz + k + x];
                    o[x] = w == 0.0f ? ec : (w == 1.0f ? v : 1.0f / (w / v + (1.0f - w) * inv_ec));
                }
            }
            __stcs(dst + f, make_float4(o[0], o[1], o[2], o[3]));
        }
    }
}

}  // namespace epsgrad
